/* pulse.h - C-ABI of the B200-native PULSE skip-local pipeline stage.
 *
 * What a "stage" is: PAPER.md:L91 (sec. III) "we allocate local buffers for skip
 * activations and their gradients. Skip activations are stored locally during the
 * forward pass, and these values are retrieved for gradient computation in the
 * backward pass"; PAPER.md:L142 (sec. IV-B) the model is a linear sequence of
 * operations whose I/O carries "an additional field for storing skip connections";
 * PAPER.md:L144 a stage pair = encoder-side ops plus the decoder-side ops that
 * consume their skips, on one device; PAPER.md:L255 (sec. VI) activations (and so the
 * skips) of every in-flight microbatch stay resident until its backward.
 * Block math (GroupNorm, SiLU, temb add, 3x3 conv, residual, concat with the cached
 * skip) is fixed by BASELINE.json north_star; formulas in SURVEY.md 8c / DESIGN.md.
 *
 * Conventions
 *  - Every call returns pulse_status_t (0 = OK), never throws/aborts/prints;
 *    pulse_last_error() gives a thread-local message.  Out-params are written only
 *    on success.
 *  - "d_" pointers are DEVICE pointers, owned by the caller (the library never
 *    allocates device memory); all must be 256-byte aligned.  Other pointers are host.
 *  - Work is enqueued on the caller's stream (a cudaStream_t passed as void*); forward
 *    and backward never synchronise the host.
 *  - Activations are NHWC in the stage dtype (fp32 or bf16).  Conv weights are
 *    [Cout][kh][kw][Cin], linear weights [out][in], all parameters in the stage dtype,
 *    packed into one buffer at the offsets pulse_stage_param_info reports.  Parameter
 *    gradients are always fp32, packed likewise.
 *  - A handle is not thread-safe; distinct handles are independent.
 */
#ifndef PULSE_H_
#define PULSE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  PULSE_OK = 0,
  PULSE_ERR_INVALID_ARG = 1,      /* null / misaligned pointer, bad enum value */
  PULSE_ERR_SHAPE = 2,            /* descriptor inconsistent (pops more than pushed, C % groups != 0 ...) */
  PULSE_ERR_UNSUPPORTED = 3,
  PULSE_ERR_BUFFER_TOO_SMALL = 4,
  PULSE_ERR_CACHE = 5,            /* slot busy / unknown microbatch / cache full */
  PULSE_ERR_STATE = 6,            /* params / workspace not bound, backward without forward */
  PULSE_ERR_CUDA = 7
} pulse_status_t;

enum { PULSE_F32 = 0, PULSE_BF16 = 1 };
enum { PULSE_OP_CONV_IN = 0, PULSE_OP_RESBLOCK = 1, PULSE_OP_DOWN = 2, PULSE_OP_UP = 3, PULSE_OP_HEAD = 4,
       PULSE_OP_ATTN = 5 /* self-attention block: GroupNorm -> 1x1 conv to q|k|v -> softmax(q k^T / sqrt(d)) v
                            per head over the H W pixels -> 1x1 conv, + residual; cin == cout, heads | cin */,
       PULSE_OP_TBLOCK = 6 /* transformer block with an optional long skip:
                              [x = Linear(concat_C(x, skip)) where skip_channels > 0 ("concat + Linear")];
                              x = x + proj(attention(qkv(LayerNorm(x)))); x = x + fc2(GELU(fc1(LayerNorm(x)))), fc1: c -> 4c;
                              tokens = the H W pixels, Linear = 1x1 conv; cin == cout, heads | cin; takes no timestep input */ };
enum { PULSE_LINK_OPEN = 0, PULSE_LINK_CLOSED = 1 };
enum { PULSE_TEMB_SINUSOIDAL = 0, PULSE_TEMB_MLP = 1 };
/* stage flags (cross-checks: same arithmetic, different kernel / summation order) */
enum {
  PULSE_FLAG_FORCE_SIMT = 1,    /* CUDA-core fp32-accumulate convs even for bf16 */
  PULSE_FLAG_GN_TWO_PASS = 2,   /* GroupNorm backward always as reduction pass + apply pass (never the one-pass
                                   cluster kernel) */
  PULSE_FLAG_CONV_PAIR = 4,     /* tcgen05 convs: the CTA-pair kernel (conv_tc2_k) wherever it covers the shape */
  PULSE_FLAG_CONV_1CTA = 8,     /* tcgen05 convs: the single-CTA kernel (conv_tc_k) wherever it covers the shape */
  /* Upsample + conv (row a6).  Default: forward and input gradient through the materialised upsampled tensor, weight
   * gradient in the 4-phase form (4/9 of the FLOPs, exact: it reads the original bf16 operands).  The 4-phase forward and
   * input gradient need PRE-SUMMED bf16 weights, one extra rounding of the weights that costs as much as one more bf16
   * store of the activations: faster (configs[2]: -5 %), but opt-in because tensors that sit just
   * under north_star's 2e-2 bar then cross it. */
  PULSE_FLAG_UP_MATERIALISED = 16, /* weight gradient through the materialised tensor too (the oracle's form everywhere) */
  PULSE_FLAG_UP_PHASE_FWD = 32,    /* forward in the 4-phase form (no upsampled tensor is written) */
  PULSE_FLAG_UP_PHASE_DGRAD = 64,  /* input gradient in the 4-phase form (one 16-tap conv over the gradient's parity view) */
  /* Pipeline execution: the encoder half and the decoder half of an OPEN stage
   * run as separate calls (pulse_stage_forward_enc / _dec, pulse_stage_backward_dec / _enc), with other microbatches'
   * halves in between.  The gradient buffers of the cached skips then live per in-flight microbatch ("local
   * buffers for skip activations and their gradients"), beside its skip-cache slot, instead of once per stage. */
  PULSE_FLAG_SPLIT = 128
};
/* kernel selector of the single-operator conv calls */
enum { PULSE_CONV_AUTO = 0, PULSE_CONV_SIMT = 1, PULSE_CONV_TC_PAIR = 2, PULSE_CONV_TC_1CTA = 3 };

/* Environment toggles (part of the library's observable behaviour; read ONCE per process at first use; none changes
 * results beyond the order of fp32 sums):
 *   PULSE_NO_PDL=1           ordinary stream-ordered launches instead of programmatic dependent launch
 *   PULSE_NO_SIDE_STREAM=1   weight gradients / shortcut convs / timestep path on the caller's stream (no fork / join)
 *   PULSE_NO_GN_FUSED=1      as PULSE_FLAG_GN_TWO_PASS, for every stage of the process
 *   PULSE_CONV_1CTA=1        as PULSE_FLAG_CONV_1CTA, for every conv of the process without an explicit selector
 *   PULSE_CONV_1CTA_TILES=k  convs with at most k single-CTA tiles take the single-CTA kernel (default: the SM count)
 *   PULSE_WGRAD_1CTA=1       single-CTA tcgen05 weight-gradient kernel everywhere
 *   PULSE_NO_SPLIT_K=1       no cluster split-K in the CTA-pair conv kernel (few-tile convs then take the single-CTA kernel) */

/* One operation of the linearised model.  cin excludes the popped skip:
 * a decoder ResBlock runs on concat_C(h[cin], skip[skip_channels]), h first. */
typedef struct {
  int kind;           /* PULSE_OP_* */
  int cin, cout;
  int skip_channels;  /* decoder ResBlock: channels of the skip it pops (LIFO); else 0 */
  int push_skip;      /* encoder op: 1 = its output goes to the skip cache */
  int heads;          /* PULSE_OP_ATTN: number of heads (head h owns channels [h d, (h+1) d), d = cin / heads); else 0 */
} pulse_op_desc;

typedef struct {
  int dtype;                         /* PULSE_F32 | PULSE_BF16 */
  int n, h, w, c_in;                 /* x_in is [n,h,w,c_in] */
  int groups; float eps;             /* GroupNorm */
  int temb_kind, temb_d0, temb_dim;  /* sinusoidal(d0) [-> MLP d0->dim->dim]; dim = T */
  int link;                          /* OPEN: h_in/e_out cross the boundary; CLOSED: h := mid(enc output) */
  int x_in_is_skip;                  /* 1 = x_in itself is pushed first */
  int n_enc_ops; const pulse_op_desc* enc_ops;
  int n_mid_ops; const pulse_op_desc* mid_ops;   /* ResBlocks only; CLOSED only */
  int n_dec_ops; const pulse_op_desc* dec_ops;
  int max_inflight;                  /* microbatches forwarded but not yet backwarded */
  unsigned flags;
} pulse_stage_desc;

typedef struct pulse_stage pulse_stage_t;
typedef struct pulse_skip_cache pulse_skip_cache_t;

/* ---- stage life cycle ----------------------------------------------------------- */
/* Validates the op lists (every skip pushed is popped exactly once, channel counts
 * chain, C % groups == 0 ...) -> PULSE_ERR_SHAPE otherwise.  The descriptor is copied. */
pulse_status_t pulse_stage_create(const pulse_stage_desc* desc, pulse_stage_t** out);
pulse_status_t pulse_stage_destroy(pulse_stage_t* stage);

/* Parameters, in the fixed order temb MLP (w1,b1,w2,b2), then per op of enc, mid, dec:
 * ResBlock: gn1.gamma gn1.beta conv1.w conv1.b temb.w temb.b gn2.gamma gn2.beta conv2.w
 * conv2.b [sc.w sc.b if cin+skip != cout]; conv_in/down/up: conv.w conv.b; head: gn.gamma
 * gn.beta conv.w conv.b; attention: gn.gamma gn.beta qkv.w [3c][1][1][c] qkv.b proj.w [c][1][1][c] proj.b;
 * transformer block: [skip.w [c][1][1][c+skip] skip.b] ln1.gamma ln1.beta qkv.w qkv.b proj.w proj.b ln2.gamma ln2.beta
 * fc1.w [4c][1][1][c] fc1.b fc2.w [c][1][1][4c] fc2.b.  name points into the handle (valid until destroy). */
pulse_status_t pulse_stage_param_count(const pulse_stage_t* stage, int* count);
pulse_status_t pulse_stage_param_info(const pulse_stage_t* stage, int index, const char** name, int* rank,
                                      int shape[4], size_t* offset_bytes, size_t* grad_offset_bytes);
pulse_status_t pulse_stage_param_bytes(const pulse_stage_t* stage, size_t* param_bytes, size_t* grad_bytes);
/* d_params: param_bytes in the stage dtype; d_grads: grad_bytes of fp32.  Both stay
 * caller-owned and must outlive the calls that use them. */
pulse_status_t pulse_stage_bind_params(pulse_stage_t* stage, const void* d_params, float* d_grads);

/* Scratch: per_stage bytes (gradient temporaries, skip-gradient buffers, reduction
 * scratch) + max_inflight * per_inflight_stash bytes (forward intermediates kept for
 * the backward of each in-flight microbatch).  Bind one buffer of at least that sum. */
pulse_status_t pulse_stage_workspace_bytes(const pulse_stage_t* stage, size_t* per_stage, size_t* per_inflight_stash);
pulse_status_t pulse_stage_bind_workspace(pulse_stage_t* stage, void* d_workspace, size_t bytes);

/* ---- skip cache (PAPER.md:L91 local skip buffers; L255 one set per in-flight microbatch) */
pulse_status_t pulse_skip_cache_bytes(const pulse_stage_t* stage, size_t* bytes_per_slot);
/* d_mem: slots * bytes_per_slot bytes.  slots must be <= desc.max_inflight. */
pulse_status_t pulse_skip_cache_create(pulse_stage_t* stage, void* d_mem, size_t bytes, int slots,
                                       pulse_skip_cache_t** out);
/* Skip k (push order) of live microbatch mb_id: device pointer and NHWC shape. */
pulse_status_t pulse_skip_cache_get(const pulse_skip_cache_t* cache, int64_t mb_id, int k, void** d_ptr, int shape[4]);
pulse_status_t pulse_skip_cache_count(const pulse_skip_cache_t* cache, int* skips_per_slot);
/* Normally implicit at the end of pulse_stage_backward. */
pulse_status_t pulse_skip_cache_release(pulse_skip_cache_t* cache, int64_t mb_id);
pulse_status_t pulse_skip_cache_stats(const pulse_skip_cache_t* cache, int* live_slots, size_t* live_bytes,
                                      size_t* peak_bytes);
pulse_status_t pulse_skip_cache_destroy(pulse_skip_cache_t* cache);

/* ---- the hot path ----------------------------------------------------------------- */
/* Forward of microbatch mb_id: acquires a free slot
 * (PULSE_ERR_CACHE if mb_id is already live or no slot is free).
 *  d_x_in  [n,h,w,c_in]                     stage dtype
 *  d_h_in  OPEN: input of the first decoder op; CLOSED: NULL
 *  d_temb  [n,temb_dim] fp32 (the embedding after the MLP; see pulse_temb_forward)
 *  d_e_out OPEN: last encoder output (written); CLOSED: NULL
 *  d_d_out last decoder output (written) */
pulse_status_t pulse_stage_forward(pulse_stage_t* stage, pulse_skip_cache_t* cache, int64_t mb_id,
                                   const void* d_x_in, const void* d_h_in, const float* d_temb,
                                   void* d_e_out, void* d_d_out, void* stream);
/* Backward of a live microbatch (rows a8-a11); releases its slot.
 *  d_g_d_out  gradient of d_out (stage dtype)
 *  d_g_e_out  OPEN: gradient of e_out or NULL (= zeros); CLOSED: NULL
 *  d_g_x_in   written if non-NULL
 *  d_g_h_in   OPEN: written; CLOSED: NULL
 *  d_g_temb   [n,temb_dim] fp32, accumulated (+=) if non-NULL
 *  accumulate_wgrad 0: parameter gradients overwritten, 1: += (fp32, row a11) */
pulse_status_t pulse_stage_backward(pulse_stage_t* stage, pulse_skip_cache_t* cache, int64_t mb_id,
                                    const void* d_g_d_out, const void* d_g_e_out, void* d_g_x_in,
                                    void* d_g_h_in, float* d_g_temb, int accumulate_wgrad, void* stream);

/* The two halves of an OPEN stage as separate calls (needs PULSE_FLAG_SPLIT; row f2): on a pipeline, the stages further in
 * run between the encoder half and the decoder half of a microbatch, and between the backward of its decoder half and of
 * its encoder half.  Order per microbatch: forward_enc (takes the slot) -> forward_dec -> backward_dec -> backward_enc
 * (releases the slot); halves of other live microbatches may run anywhere in between.  Arguments as in the one-call
 * forms.  accumulate_wgrad applies to backward_dec (0: zero the parameter gradients first); backward_enc always adds. */
pulse_status_t pulse_stage_forward_enc(pulse_stage_t* stage, pulse_skip_cache_t* cache, int64_t mb_id, const void* d_x_in,
                                       const float* d_temb, void* d_e_out, void* stream);
pulse_status_t pulse_stage_forward_dec(pulse_stage_t* stage, pulse_skip_cache_t* cache, int64_t mb_id, const void* d_h_in,
                                       void* d_d_out, void* stream);
pulse_status_t pulse_stage_backward_dec(pulse_stage_t* stage, pulse_skip_cache_t* cache, int64_t mb_id,
                                        const void* d_g_d_out, void* d_g_h_in, float* d_g_temb, int accumulate_wgrad,
                                        void* stream);
pulse_status_t pulse_stage_backward_enc(pulse_stage_t* stage, pulse_skip_cache_t* cache, int64_t mb_id,
                                        const void* d_g_e_out, void* d_g_x_in, float* d_g_temb, void* stream);

/* The same two calls with the timestep path inside (rows a1, a7), so that it runs beside the chain instead of
 * before / after it: forward = pulse_temb_forward(d_t -> d_emb, d_temb_stash) + pulse_stage_forward(d_temb = d_emb);
 * backward = pulse_stage_backward + pulse_temb_backward(d_g_temb, d_temb_stash).  Same results as the separate
 * calls.  d_emb [n,temb_dim] fp32 and d_temb_stash (pulse_temb_stash_elems floats) are written by the forward and
 * kept by the caller until the backward of the microbatch; d_g_temb must be zeroed by the caller (it is +=). */
pulse_status_t pulse_stage_forward_temb(pulse_stage_t* stage, pulse_skip_cache_t* cache, int64_t mb_id,
                                        const void* d_x_in, const void* d_h_in, const int64_t* d_t, float* d_emb,
                                        float* d_temb_stash, void* d_e_out, void* d_d_out, void* stream);
pulse_status_t pulse_stage_backward_temb(pulse_stage_t* stage, pulse_skip_cache_t* cache, int64_t mb_id,
                                         const void* d_g_d_out, const void* d_g_e_out, void* d_g_x_in,
                                         void* d_g_h_in, float* d_g_temb, const float* d_temb_stash,
                                         int accumulate_wgrad, void* stream);

/* ---- helpers on the path (row a1, a7) ----------------------------------------------- */
/* emb0 = [cos(t f_i), sin(t f_i)], f_i = exp(-ln(1e4) i/half); MLP kind: emb = W2 SiLU(W1 emb0 + b1) + b2
 * using the bound temb.* parameters.  d_t: int64 [n].  d_emb: fp32 [n,temb_dim].
 * d_stash: fp32 scratch of pulse_temb_stash_elems floats kept by the caller until
 * pulse_temb_backward of the same microbatch. */
pulse_status_t pulse_temb_stash_elems(const pulse_stage_t* stage, size_t* elems);
pulse_status_t pulse_temb_forward(pulse_stage_t* stage, const int64_t* d_t, float* d_emb, float* d_stash, void* stream);
/* Gradients of temb.w1/b1/w2/b2 from d_g_emb [n,temb_dim] (no-op for the sinusoidal kind). */
pulse_status_t pulse_temb_backward(pulse_stage_t* stage, const float* d_g_emb, const float* d_stash,
                                   int accumulate_wgrad, void* stream);
/* L = scale * mean((d - target)^2) added into *d_loss (fp32, caller zeroes it);
 * g_d = scale * 2 (d - target) / numel in dtype. */
pulse_status_t pulse_mse_fwd_bwd(int dtype, const void* d_d, const void* d_target, size_t numel, float scale,
                                 float* d_loss, void* d_g_d, void* stream);

/* ---- single operators (the kernels of rows a2/a4/a5/a6/a8-a10 in isolation; used by the
 * kernel-level parity tests and microbenchmarks).  NHWC activations, weights [cout][k][k][cin],
 * k in {1,3}, pad (k-1)/2, stride in {1,2}; dtype as above.  kernel: PULSE_CONV_AUTO (tcgen05 where the shape is
 * covered - CTA-pair or single-CTA kernel by tile count - else CUDA cores), PULSE_CONV_SIMT (CUDA cores),
 * PULSE_CONV_TC_PAIR / PULSE_CONV_TC_1CTA (that tcgen05 kernel; PULSE_ERR_UNSUPPORTED if it does not cover the
 * shape / dtype).  SURVEY.md 8c item 2. */
/* out[n,y,x,co] = bias[co] + pn[n,co] + residual[n,y,x,co] + sum W[co][r][s][c] in[n, y st+r-pad, x st+s-pad, c],
 * in = concat_C(src0[c0], src1[c1]) (src1 may be NULL with c1 = 0); bias/pn/residual may be NULL.
 * d_chan_stats (nullable): [n][2][cout] fp32, += the per-(image, channel) sum and sum of squares over the pixels of
 * the STORED output - the statistics hand-off to the GroupNorm that reads this tensor (caller zeroes it).  The
 * CTA-pair kernel emits them from its epilogue; for the other kernels a statistics pass follows the conv.  (For
 * PULSE_F32 tensors the sums are taken about a pivot, x - x[n, pixel 0, c], reading R22; they are an
 * opaque hand-off to pulse_groupnorm_silu either way.) */
pulse_status_t pulse_conv2d(int dtype, int kernel, const void* d_src0, int c0, const void* d_src1, int c1,
                            int n, int h, int w, int ksize, int stride, const void* d_w, int cout,
                            const void* d_bias, const float* d_pn, const void* d_residual, void* d_out,
                            float* d_chan_stats, void* stream);
/* g_in[n,h,w,cin] (+)= adjoint of the conv in its input, from g [n,hout,wout,cout].
 * d_wt_scratch: cout*k*k*cin elements of dtype (holds the flipped/transposed weights). */
pulse_status_t pulse_conv2d_dgrad(int dtype, int kernel, const void* d_g, int n, int h, int w, int cin,
                                  int ksize, int stride, const void* d_w, int cout, void* d_wt_scratch,
                                  void* d_g_in, int accumulate, void* stream);
/* dw[cout][k][k][c0+c1] (+)= sum_{n,y,x} g[n,y,x,co] in[n, y st+r-pad, x st+s-pad, c]  (fp32).
 * accumulate = 1: added to what d_dw holds.  accumulate = 0: d_dw is overwritten, whatever it held - stored directly
 * where the tcgen05 kernel owns whole output tiles (many tiles, few pixels: the deep UNet levels), zeroed by the call
 * and added into otherwise. */
pulse_status_t pulse_conv2d_wgrad(int dtype, int force_simt, const void* d_src0, int c0, const void* d_src1, int c1,
                                  int n, int h, int w, int ksize, int stride, const void* d_g, int cout,
                                  float* d_dw, int accumulate, void* stream);

/* Nearest-2x upsample followed by a 3x3 pad-1 conv (row a6), computed WITHOUT the upsampled tensor:
 * output pixel (2y+py, 2x+px) is a 2x2 conv of the low-resolution input with the pre-summed weights of its parity phase
 * (4 taps on h x w pixels per phase instead of 9 taps on 2h x 2w: 4/9 of the FLOPs; the result equals
 * conv3x3(upsample2(src)) up to the rounding of the pre-summed bf16 weights).  bf16 / tcgen05 only; kernel: PULSE_CONV_AUTO,
 * _TC_PAIR or _TC_1CTA.  src [n,h,w,cin], w [cout][3][3][cin], out [n,2h,2w,cout].
 * d_wp_scratch / d_wpt_scratch: 16*cout*cin elements of dtype (the pre-summed phase weights, written by the call).
 * dgrad: g [n,2h,2w,cout] -> g_in [n,h,w,cin] (written).  wgrad: dw [cout][3][3][cin] fp32, accumulated. */
pulse_status_t pulse_upsample_conv2d(int dtype, int kernel, const void* d_src, int n, int h, int w, int cin,
                                     const void* d_w, int cout, const void* d_bias, void* d_wp_scratch, void* d_out,
                                     float* d_chan_stats, void* stream);
pulse_status_t pulse_upsample_conv2d_dgrad(int dtype, int kernel, const void* d_g, int n, int h, int w, int cin,
                                           const void* d_w, int cout, void* d_wpt_scratch, void* d_g_in, void* stream);
pulse_status_t pulse_upsample_conv2d_wgrad(int dtype, const void* d_src, int n, int h, int w, int cin, const void* d_g,
                                           int cout, float* d_dw, void* stream);

/* Scaled dot-product self-attention in isolation (the core of PULSE_OP_ATTN):
 *   S = q k^T / sqrt(d), P = softmax over keys, o = P v, per (image, head), d = c / heads <= 128.
 * d_qkv [n][tokens][3c]: q | k | v interleaved per token as the 1x1 conv leaves them (head h = channels [h d, (h+1) d)
 * of each third); d_o, d_g_o [n][tokens][c]; d_g_qkv as d_qkv (written).  d_stats: pulse_attention_stats_floats(n,
 * heads, tokens) fp32, written by the forward (log-sum-exp per query) and the backward, kept between the two.
 * The T x T matrix is never written; no atomics.  bf16 tensors with 64 or 128 channels per head take the tcgen05
 * kernels (Q K^T, P V and the five products of the backward on the tensor cores, softmax and its Jacobian in fp32 on the
 * TMEM accumulator rows, P / g_S handed over as bf16) unless force_simt != 0; everything else takes CUDA-core kernels
 * with fp32 arithmetic on fp32 or bf16 storage. */
size_t pulse_attention_stats_floats(int n, int heads, int tokens);
pulse_status_t pulse_attention(int dtype, int force_simt, const void* d_qkv, int n, int tokens, int c, int heads, void* d_o,
                               float* d_stats, void* stream);
pulse_status_t pulse_attention_backward(int dtype, int force_simt, const void* d_qkv, const void* d_g_o, int n, int tokens,
                                        int c, int heads, float* d_stats, void* d_g_qkv, void* stream);

/* GroupNorm + SiLU in isolation (the kernels of rows a2/a5 and a8/a9), on
 * x = concat_C(x0[c0], x1[c1]) (x1 may be NULL with c1 = 0), NHWC, C = c0 + c1 divisible by groups
 * (a group may straddle the x0|x1 boundary):
 *   mu, var per (image, group) over its C/groups channels and all pixels (biased variance),
 *   r = 1/sqrt(var + eps), xhat = (x - mu) r, y = gamma xhat + beta, a = y sigmoid(y).
 * d_stats: caller-owned fp32 scratch of pulse_groupnorm_stats_floats(n, C, groups) elements; the forward
 * fills it (per-(image, channel) sums, then mean / r per (image, group)) and the backward of the same
 * tensor reads it.  reuse_stats != 0: d_stats already holds the statistics of this x (an earlier forward
 * call): only the normalise + SiLU pass runs (what a conv epilogue that emitted the sums leaves to do).
 * gamma, beta: [C] in dtype.  d_a: [n,h,w,C].  Errors: PULSE_ERR_INVALID_ARG (null pointer, sizes <= 0,
 * dtype), PULSE_ERR_SHAPE (C % groups, channel counts not a multiple of the 16-byte vector: 4 fp32 / 8 bf16). */
size_t pulse_groupnorm_stats_floats(int n, int c, int groups);
pulse_status_t pulse_groupnorm_silu(int dtype, const void* d_x0, int c0, const void* d_x1, int c1, int n, int h, int w,
                                    int groups, float eps, const void* d_gamma, const void* d_beta, float* d_stats,
                                    int reuse_stats, void* d_a, void* stream);
/* Backward of the above from g_a [n,h,w,C]:
 *   g_y = g_a SiLU'(y); dgamma += sum g_y xhat; dbeta += sum g_y (fp32 [C], accumulated: caller zeroes);
 *   q = gamma g_y; A = mean_S q; B = mean_S q xhat; g_x = r (q - A - xhat B) + add,
 * add: [n,h,w,C] in dtype or NULL.  g_x is split at c0: channels [0,c0) -> d_g_x0 [n,h,w,c0], the rest ->
 * d_g_x1 [n,h,w,c1] (the skip-gradient buffer of PAPER.md:L91); accumulate0 / accumulate1 != 0: += into that
 * destination.  d_stats: as the forward left it.  d_scratch: n*2*C fp32 (zeroed here; used by the two-kernel
 * form).  two_pass != 0 forces the two-kernel form (reduction pass + apply pass) where the one-pass cluster
 * kernel would apply (bf16 tensors whose per-image group slices fit a cluster's shared memory).
 * fwd_data_ready: 0 = the call is ordered after everything enqueued on the stream before it (it may directly follow
 * the pulse_groupnorm_silu that writes d_stats); nonzero = the caller guarantees that x0 / x1 and d_stats were
 * complete before the PREVIOUS kernel of the stream started (as inside a stage, where they are forward-pass data):
 * the one-pass kernel is then launched with programmatic serialization and prefetches them during that kernel's tail. */
pulse_status_t pulse_groupnorm_silu_backward(int dtype, int two_pass, int fwd_data_ready, const void* d_g_a, const void* d_x0, int c0,
                                             const void* d_x1, int c1, int n, int h, int w, int groups, float eps,
                                             const void* d_gamma, const void* d_beta, const float* d_stats,
                                             float* d_scratch, const void* d_add, void* d_g_x0, int accumulate0,
                                             void* d_g_x1, int accumulate1, float* d_dgamma, float* d_dbeta,
                                             void* stream);

/* ---- skip-aware balanced partitioning (host code, no device work) -------------------------
 * PAPER.md:L140-L197 (sec. IV-B, Eq. 1-5, Alg. 1): cut the linear sequence of n_ops operations into p stages (p even;
 * stage q and stage p-q+1 share a device) such that both ends of every skip connection (skip_src[s] < skip_dst[s],
 * 1-based operation indices, |src - dst| > 1) lie in a collocated stage pair, minimising the slowest stage
 *   max_m ( sum_{l in S_m} t_f[l] + lambda (t_lat + M_a / b_inter) ),
 * M_a = act_bytes of the stage's last operation (encoder side) or of the operation before its first (decoder side),
 * Eq. 2-3.  t_f, act_bytes: host arrays [n_ops] (act_bytes may be NULL when lambda == 0).
 * cuts [p-1] (host, written): 1-based index of the last operation of stages 1 .. p-1; *bottleneck: the optimum.
 * O(p n^3) time, O(p n^2) memory.  PULSE_ERR_SHAPE: no feasible partition / bad skip indices. */
pulse_status_t pulse_partition(int n_ops, const double* t_f, const double* act_bytes, int n_skips, const int* skip_src,
                               const int* skip_dst, int p, double lambda, double t_lat, double b_inter, int* cuts,
                               double* bottleneck);

/* ---- per-kernel-class timing (row d: measurement) -------------------------------------------
 * With profiling enabled, forward/backward bracket every kernel of these classes with CUDA events
 * on the caller's stream: 0 tcgen05 conv (fprop+dgrad), 1 tcgen05 wgrad, 2 CUDA-core conv/wgrad,
 * 3 GroupNorm+SiLU forward, 4 GroupNorm+SiLU backward, 5 everything else.  pulse_stage_profile_read
 * synchronises those events and returns, per class, total milliseconds, launches, algorithmic FLOPs
 * (2*M*N*K of the convs) and algorithmic bytes, then clears the records. */
enum { PULSE_KCLASS_CONV_TC = 0, PULSE_KCLASS_WGRAD_TC = 1, PULSE_KCLASS_CONV_SIMT = 2, PULSE_KCLASS_GN_FWD = 3,
       PULSE_KCLASS_GN_BWD = 4, PULSE_KCLASS_OTHER = 5, PULSE_KCLASS_COUNT = 6 };
pulse_status_t pulse_stage_profile(pulse_stage_t* stage, int enable);
pulse_status_t pulse_stage_profile_read(pulse_stage_t* stage, double ms[6], uint64_t launches[6], double flops[6],
                                        double bytes[6]);

/* Number of kernels this handle has launched so far (bench.py "gpu_launches"). */
pulse_status_t pulse_stage_launch_count(const pulse_stage_t* stage, uint64_t* launches);

int pulse_version(void);
const char* pulse_status_string(pulse_status_t s);
const char* pulse_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* PULSE_H_ */
