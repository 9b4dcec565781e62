// kernels.h - host launchers of the CUDA kernels (internal to libpulse.so).
// Every launcher enqueues on `st`, returns the number of kernels it launched.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

namespace pulse {

enum { DT_F32 = 0, DT_BF16 = 1 };
static inline size_t dt_size(int dt) { return dt == DT_F32 ? 4 : 2; }

// Channel concat of two NHWC tensors with equal N,H,W (the "virtual concat": PAPER.md
// L91 skip buffer read in place, north_star "concat fused into the operand loader").
struct Cat {
  const void* p0; int c0;
  const void* p1; int c1;     // p1 == nullptr, c1 == 0 for a single source
  int c() const { return c0 + c1; }
};

// ---- GroupNorm + SiLU -------------------------------------------
// Statistics interface: "channel stats" cst[n][2][c] fp32 = per-(image, channel) sum and sum of squares over
// the pixels of ONE tensor, accumulated with atomics (zero them first).  Produced by chan_stats (or, later, by
// the conv epilogue that writes the tensor), consumed by every GroupNorm site that reads the tensor; a dual-
// source site takes one cst per source.
struct RowPlan { int tpr, rows, nchunks; };
RowPlan row_plan(int dt, int hw, int c, int n, int max_threads);
// copy (nullable): the same pass also copies x there (a tensor that enters the stage is stashed and measured at once)
int chan_stats(int dt, const void* x, int n, int hw, int c, float* cst, cudaStream_t st, void* copy = nullptr);
// mr_out: [n][2][groups] fp32, the group means and reciprocal standard deviations, kept for the backward
int gn_silu_fwd(int dt, Cat x, int n, int hw, int groups, float eps, const void* gamma, const void* beta,
                const float* cst0, const float* cst1, float* mr_out, void* a_out, cudaStream_t st, int act = 1);
// act = 0 (here and in the backward launchers): plain GroupNorm, y = gamma xhat + beta, no SiLU (attention blocks)
// g_x = r(gamma g_y - A - xhat B) [+ add]; channels [0,dc0) -> dst0, rest -> dst1; accX: += instead of =
// bst: [n][2][C] fp32 scratch, zeroed by the caller (per-(image, channel) sums of g_y and g_y xhat).
// dgamma/dbeta: fp32, +=.  cs0/cs1 (nullable): [n][dc0] / [n][C-dc0] fp32, += the per-(image, channel) pixel
// sums of what this call adds to dst0 / dst1 (bias and temb-projection gradients are made of these).
int gn_silu_bwd(int dt, const void* g_a, Cat x, int n, int hw, int groups, float eps, const void* gamma,
                const void* beta, const float* mr, float* bst, const void* add, void* dst0,
                int dc0, int acc0, void* dst1, int acc1, float* dgamma, float* dbeta, float* cs0, float* cs1,
                cudaStream_t st, bool allow_fused = true, bool fwd_data_ready = true, int act = 1);

// the same in one launch (norm_fused.cu; bf16, mean / rstd from the forward); 0 = shape not covered, nothing launched.
// fwd_data_ready: x and mr were complete before the PREVIOUS kernel of the stream started (true inside a stage: they
// are forward-pass data), so the kernel may read them before its dependency wait; false: launched without
// programmatic serialization (the single-operator entry point, where the forward may be the previous kernel).
int gn_bwd_fused(const void* g_a, Cat x, int n, int hw, int groups, const void* gamma, const void* beta, const float* mr,
                 const void* add, void* dst0, int dc0, int acc0, void* dst1, int acc1, float* dgamma, float* dbeta,
                 float* cs0, float* cs1, cudaStream_t st, bool fwd_data_ready = true, int act = 1);

// ---- attention core (attention.cu) ------------------------------------
// qkv [n][T][3C] (q | k | v per pixel, head h = channels [h d, (h+1) d) of each third), o / g_o [n][T][C];
// stats: attn_stats_floats(n, heads, T) floats (log-sum-exp of the scaled scores, then D = rowsum(P g_P)) written by the
// forward / backward and kept between them
bool attn_supported(int C, int heads);
size_t attn_stats_floats(int n, int heads, int T);
// use_tc: the tcgen05 forward (attention_tc.cu) where it applies (bf16, 64 or 128 channels per head), else CUDA cores
int attn_fwd(int dt, const void* qkv, int n, int T, int C, int heads, void* o, float* stats, cudaStream_t st, bool use_tc = true);
bool attn_fwd_tc_supported(int dt, int C, int heads);
int attn_fwd_tc(const void* qkv, int n, int T, int C, int heads, void* o, float* lse, cudaStream_t st);
int attn_bwd(int dt, const void* qkv, const void* g_o, int n, int T, int C, int heads, float* stats, void* g_qkv,
             cudaStream_t st, bool use_tc = true);
int attn_bwd_tc(const void* qkv, const void* g_o, int n, int T, int C, int heads, float* stats, void* g_qkv, cudaStream_t st);

// ---- transformer-block pointwise kernels (tblock.cu) ------------------------
// LayerNorm over the C channels of each of `tokens` rows; stat [tokens][2] fp32 = mean, rstd (written by the forward)
int layernorm_fwd(int dt, const void* x, size_t tokens, int C, float eps, const void* gamma, const void* beta, float* stat,
                  void* y, cudaStream_t st);
// g_x (+)= r (q - mean q - xhat mean(q xhat)) [+ add], q = g_y gamma; dgamma / dbeta: fp32, +=
int layernorm_bwd(int dt, const void* g_y, const void* x, size_t tokens, int C, const void* gamma, const float* stat,
                  const void* add, void* g_x, int acc, float* dgamma, float* dbeta, cudaStream_t st);
int gelu_fwd(int dt, const void* x, void* y, size_t numel, cudaStream_t st);
int gelu_bwd(int dt, const void* x, const void* g, void* g_x, size_t numel, cudaStream_t st);     // g_x = g GELU'(x)

// ---- small ops -----------------------------------------------------------------------
// cs[n][c] += sum over pixels of g[n][hw][c]   (tensors whose writers could not emit their column sums)
int colsum(int dt, const void* g, int n, int hw, int c, float* cs, cudaStream_t st);
// out[n][o] = sum_i W[o][i] f(in[n][i]) + b[o]; f = SiLU if silu_in.  W,b in dtype dt; in/out fp32
int linear_fwd(int dt, const float* in, int n, int din, int dout, const void* w, const void* b, int silu_in,
               float* out, cudaStream_t st);
// dW[o][i] += sum_n g[n][o] f(in[n][i]); db[o] += sum_n g[n][o];
// g_in[n][i] (+)= (sum_o g[n][o] W[o][i]) f'(in[n][i])   (g_in may be null)
int linear_bwd(int dt, const float* in, const float* g, int n, int din, int dout, const void* w, int silu_in,
               float* dw, float* db, float* g_in, int acc_g_in, cudaStream_t st);
// Batched over the ops of a stage (one launch per 16 entries instead of one per op):
struct ProjEntry { const void* w; const void* b; float* out; int cout; };          // out[n][cout] = W silu(emb) + b
int temb_proj_batch(int dt, const float* emb, int n, int T, const ProjEntry* e, int count, cudaStream_t st);
// Everything an op's small gradients need, from the column sums the big kernels emitted:
//   db_out (+ db_out2) += sum_n cs_out[n][c];  with gp (ResBlocks): db1 += sum_n gp, dtb += sum_n gp,
//   dtw[c][j] += sum_n gp[n][c] silu(emb[n][j]),  g_emb[n][j] += sum_c gp[n][c] tw[c][j] silu'(emb[n][j])
struct SmallGradEntry {
  const float* cs_out; float* db_out; float* db_out2;
  const float* gp; float* db1; float* dtb; float* dtw; const void* tw;
  int cout;
};
int small_grads_batch(int dt, const float* emb, float* g_emb, int n, int T, const SmallGradEntry* e, int count,
                      cudaStream_t st);
struct TransposeEntry { const void* w; void* wt; int cout, k, cin; };
int flip_transpose_batch(int dt, const TransposeEntry* e, int count, cudaStream_t st);
int sinusoidal(const int64_t* t, int n, int d, float* out, cudaStream_t st);
int mse_fwd_bwd(int dt, const void* d, const void* target, size_t numel, float scale, float* loss, void* g,
                cudaStream_t st);
// Wp [4][cout][4][cin] (nullable) and WpT [cin][16][cout] (nullable) of CONV_UP2 / CONV_UP2_DGRAD from W [cout][3][3][cin];
// sums in fp32, stored in dtype
int up2_weights(int dt, const void* w, int cout, int cin, void* wp, void* wpt, cudaStream_t st);
int upsample2(int dt, const void* in, int n, int h, int w, int c, void* out, cudaStream_t st);
int upsample2_bwd(int dt, const void* g_u, int n, int h, int w, int c, void* g_out, cudaStream_t st);  // h,w: low-res
int add_inplace(int dt, void* dst, const void* src, size_t numel, cudaStream_t st);
// Wt[ci][k-1-r][k-1-s][co] = W[co][r][s][ci]
int flip_transpose(int dt, const void* w, int cout, int k, int cin, void* wt, cudaStream_t st);

// ---- convolution ---------------------------------------------------
// CONV_UP2 / CONV_UP2_DGRAD: nearest-2x upsample + 3x3 conv WITHOUT the upsampled tensor:
// output pixel (2y+py, 2x+px) sees the low-resolution pixels (y+dy, x+dx), dy = a-1+py, dx = b-1+px, a,b in {0,1}, through
// the pre-summed weights Wp[2py+px][co][2a+b][ci] = sum of W[co][r][s][ci] over r in R(py,a), s in R(px,b),
// R(0,0)={0}, R(0,1)={1,2}, R(1,0)={0,1}, R(1,1)={2}  (up2_weights): 4 taps on h x w pixels per phase instead of 9 taps on
// 2h x 2w = 4/9 of the FLOPs.  The adjoint in the input is one 16-tap conv over the parity view of the gradient.
enum { CONV_FPROP = 0, CONV_DGRAD_S2 = 1, CONV_UP2 = 2, CONV_UP2_DGRAD = 3 };
enum { CONV_K_AUTO = 0, CONV_K_PAIR = 1, CONV_K_1CTA = 2 };      // which tcgen05 conv kernel (ConvArgs::kernel)
struct ConvArgs {
  int dt;
  Cat src; int n, hin, win;       // source tensor(s) [n,hin,win,c]
  int hout, wout;                 // output pixels
  int ksize, stride, mode;        // mode CONV_DGRAD_S2: src pixel = (y + r - pad)/2 when even (stride ignored)
                                  // CONV_UP2: src low-res [n,hin,win,c], out [n,2hin,2win,cout], w = Wp [4][cout][4][c]
                                  // CONV_UP2_DGRAD: src = gradient [n,hin,win,c] (high-res), out [n,hin/2,win/2,cout],
                                  //                 w = WpT [cout][16][c] (cout = the conv's input channels)
  const void* w;                  // [cout][k][k][src.c()]
  int cout;
  const void* bias;               // [cout] dtype, or null
  const float* pn;                // [n][cout] fp32 per-sample bias (temb projection), or null
  const void* residual;           // [n,hout,wout,cout] dtype, added, or null (may alias out)
  void* out; int accumulate;      // out (+)= result
  int kernel = CONV_K_AUTO;       // tcgen05 kernel choice (tests / stage flags); AUTO: by tile count
  float* cst = nullptr;           // if non-null and the kernel can (conv_emits_stats): channel stats [n][2][cout] of
                                  // the stored output are accumulated here by the epilogue (norm.cu interface)
};
bool conv_emits_stats(const ConvArgs& a);   // true: conv_tc_any(a) fills a.cst itself; false: run chan_stats after it
int conv_simt(const ConvArgs& a, cudaStream_t st);
struct WgradArgs {
  int dt;
  Cat src; int n, hin, win;       // forward input
  const void* g; int hout, wout, cout;   // forward output gradient [n,hout,wout,cout]
  int ksize, stride;
  float* dw;                      // [cout][k][k][src.c()] fp32, atomically accumulated
  int up2 = 0;                    // 1: the conv of CONV_UP2: src low-res [n,hin,win,c], g [n,2hin,2win,cout]; dw is the 9-tap gradient
  int overwrite = 0;              // 1: dw = (not +=); honoured only where wgrad_whole_tiles(a) holds (the caller zeroes otherwise)
};
// the tcgen05 pair kernel gives every output tile of dw to ONE CTA pair (many output tiles, few pixels: the deep UNet
// levels), so that it can store instead of reduce-add and dw needs no zeroing
bool wgrad_whole_tiles(const WgradArgs& a);
int wgrad_simt(const WgradArgs& a, cudaStream_t st);
// 4 channels on one side (conv_in, head; conv_thin.cu): conv_simt / wgrad_simt route to these when they apply
bool conv_thin_supported(const ConvArgs& a);
int conv_thin(const ConvArgs& a, cudaStream_t st);
bool wgrad_thin_supported(const WgradArgs& a);
int wgrad_thin(const WgradArgs& a, cudaStream_t st);

// tcgen05 / TMA path (bf16 only).  *_supported say whether the shape maps onto the tiles.
bool conv_tc_supported(const ConvArgs& a);
int conv_tc(const ConvArgs& a, cudaStream_t st);
// CTA-pair (cta_group::2) variant, 256-pixel x 320-channel tiles (conv_tc2.cu); preferred where it applies
bool conv_tc2_supported(const ConvArgs& a);
int conv_tc2(const ConvArgs& a, cudaStream_t st);
// picks conv_tc2 or conv_tc (ConvArgs::kernel, toggles.h); *_supported: false if the chosen kernel(s) do not apply
bool conv_tc_any_supported(const ConvArgs& a);
int conv_tc_any(const ConvArgs& a, cudaStream_t st);
bool wgrad_tc_supported(const WgradArgs& a);
int wgrad_tc(const WgradArgs& a, cudaStream_t st);
bool wgrad_tc2_supported(const WgradArgs& a);      // CTA-pair variant (wgrad_tc2.cu), preferred where it applies
int wgrad_tc2(const WgradArgs& a, cudaStream_t st);
bool wgrad_tc_any_supported(const WgradArgs& a);   // PULSE_WGRAD_1CTA=1 forces the single-CTA kernel
int wgrad_tc_any(const WgradArgs& a, cudaStream_t st);
const char* tc_last_error();

}  // namespace pulse
