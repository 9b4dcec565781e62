// stage.h - host-side plan of one collocated stage (internal).
#pragma once
#include <map>
#include <string>
#include <utility>
#include <vector>

#include "../../include/pulse.h"
#include "kernels.h"

namespace pulse {

enum Region { R_NONE = 0, R_SKIP = 1, R_STASH = 2, R_WORK = 3 };

struct TRef {               // an NHWC tensor [n,h,w,c] at a byte offset inside a region
  int region = R_NONE;
  size_t off = 0;
  int h = 0, w = 0, c = 0;
};

struct ParamInfo {
  std::string name;
  int rank; int shape[4];
  size_t numel, off, goff;  // byte offsets into the param (stage dtype) / grad (fp32) buffers
};

constexpr size_t NO_OFF = (size_t)-1;

struct OpPlan {
  int kind, cin, cskip, cout, heads = 0;
  int hin, win, hout, wout;
  int x0 = -1, x1 = -1, out = -1;           // indices into Stage::tensors (activations)
  int a1 = -1, h1 = -1, a2 = -1, u = -1;    // stashed intermediates
  int tx1 = -1, tl2 = -1, tf1 = -1, tg = -1; // transformer block: x1, LN2 output, fc1 output, GELU output (a1 = LN1 output,
                                            // h1 = qkv, a2 = attention output, u = Linear(concat) output)
  size_t ln1 = 0, ln2 = 0;                  // slot stash: [tokens][2] fp32 mean / rstd of the LayerNorm sites
  size_t wt3 = 0, wt4 = 0;                  // R_WORK: transposed fc1 / fc2 weights
  size_t bst1 = 0, bst2 = 0;                // R_WORK (zeroed area): GroupNorm backward sums [n][2][C] fp32 per site
  size_t gp = 0;                            // R_WORK (zeroed area): [n][cout] fp32 pixel sums of g_h1
  size_t pn = 0;                            // byte offset in the slot stash ([n,cout] fp32)
  size_t mr1 = 0, mr2 = 0;                  // slot stash: [n][2][G] fp32 group mean / rstd of the GroupNorm sites
  size_t lse = 0;                           // slot stash (attention): softmax statistics, attn_stats_floats() floats
  size_t wt1 = 0, wt2 = 0, wtsc = 0;        // R_WORK: flipped/transposed conv weights (kept across a wave)
  int p[16];                                // parameter indices (see stage.cu)
  int push = -1, pop = -1;
  // backward write modes decided at plan time (0: '=', 1: '+=')
  int acc_x0 = 0, acc_x1 = 0;
};

struct Tensor {
  TRef ref;              // forward value
  size_t goff = 0;       // gradient buffer (R_WORK; per-slot R_STASH if g_in_stash), same shape/dtype
  bool g_in_stash = false;   // PULSE_FLAG_SPLIT: gradient of a cached skip, kept per in-flight microbatch
  bool gn_input = false; // read by a GroupNorm site: carries channel stats
  size_t cst = NO_OFF;   // R_STASH (zeroed area): channel stats [n][2][c] fp32 of the forward value
  bool is_out = false;   // output of an op with a bias: its gradient's pixel sums are needed
  size_t cs = NO_OFF;    // R_WORK (zeroed area): [n][c] fp32 pixel sums of the gradient
  bool cs_fused = true;  // every writer of the gradient emits its sums (else a colsum pass runs)
};

}  // namespace pulse

pulse_status_t pulse_set_error(pulse_status_t s, const char* fmt, ...);
#define fail pulse_set_error
#define CK_CUDA(x)                                                                            \
  do {                                                                                        \
    cudaError_t e_ = (x);                                                                     \
    if (e_ != cudaSuccess) return fail(PULSE_ERR_CUDA, "%s: %s", #x, cudaGetErrorString(e_)); \
  } while (0)
// parameter slots of OpPlan::p
enum { P_GN1G = 0, P_GN1B, P_C1W, P_C1B, P_TW, P_TB, P_GN2G, P_GN2B, P_C2W, P_C2B, P_SCW, P_SCB, P_F2W, P_F2B };
// transformer block: GN1 = ln1, C1 = qkv, C2 = proj, GN2 = ln2, T = fc1, F2 = fc2, SC = the long skip's Linear

struct pulse_stage {
  pulse_stage_desc d;
  std::vector<pulse_op_desc> enc, mid, dec;
  std::vector<pulse::ParamInfo> params;
  std::map<std::string, int> pindex;
  size_t param_bytes = 0, grad_bytes = 0, temb_grad_bytes = 0;
  std::vector<pulse::Tensor> tensors;
  std::vector<pulse::OpPlan> ops;           // enc, mid, dec concatenated
  int n_enc = 0, n_mid = 0, n_dec = 0;
  std::vector<int> skip_tensor;             // push order -> tensor index
  int t_xin = -1, t_hin = -1, t_eout = -1, t_dout = -1;
  size_t skip_bytes = 0, stash_bytes = 0, work_bytes = 0;
  size_t emb_off = 0;                       // slot stash: copy of temb [n,T] fp32
  size_t cst_begin = 0, cst_end = 0;        // slot stash: channel-stats area, zeroed at the start of forward
  size_t zero_begin = 0, zero_end = 0;      // workspace: backward sums area, zeroed at the start of backward
  bool wt_valid = false;                    // transposed weights match the bound parameters
  bool eout_grad_by_dec = false;            // PULSE_FLAG_SPLIT: a decoder op writes the gradient of e_out before g_e_out arrives
  // weight-gradient tensors whose tcgen05 kernel owns whole output tiles (kernels.h wgrad_whole_tiles): byte ranges of
  // d_grads, recorded by the first backward; later first-of-a-step backwards store into them and zero only the rest
  std::vector<std::pair<size_t, size_t>> own_runs, zero_runs;
  bool own_valid = false;
  bool wp_valid = false;                    // pre-summed phase weights of the up convs (forward) match them
  // per-stage workspace offsets (bytes)
  size_t w_ga2 = 0, w_gh1 = 0, w_gh1b = 0, w_ga1 = 0, w_gsc = 0, w_gu = 0, w_tmpf = 0, w_gqkv = 0, w_t4a = 0, w_t4b = 0, w_tca = 0, w_tcb = 0;
  // weight-gradient kernels run on a side stream, concurrently with the dgrad / GroupNorm chain of the backward
  // (fork / join with events; legal inside CUDA-graph capture).  PULSE_NO_SIDE_STREAM=1 disables it.
  cudaStream_t side = nullptr;
  cudaStream_t side2 = nullptr;             // the tail of the backward (bias / temb gradients, timestep-MLP backward)
  std::vector<cudaEvent_t> sync_events;
  int side_mode = -1;                       // -1 unknown, 0 off, 1 on
  bool last_was_backward = true;            // a forward that follows a backward starts a new step: weights may have changed
  const char* d_params = nullptr; float* d_grads = nullptr;
  char* d_work = nullptr; size_t work_bound = 0;
  uint64_t launches = 0;
  // profiling (pulse_stage_profile): event pairs per kernel-class span
  struct Span { int klass; cudaEvent_t e0, e1; double flops, bytes; int launches; };
  bool profiling = false;
  std::vector<Span> spans;
  std::vector<cudaEvent_t> event_pool;
  size_t esz() const { return d.dtype == PULSE_F32 ? 4 : 2; }
};

struct pulse_skip_cache {
  pulse_stage* stage;
  char* base; int slots; size_t bytes_per_slot;
  std::vector<int64_t> mb;     // microbatch id per slot, -1 = free
  std::vector<int> phase;      // split calls: 1 forward_enc done, 2 forward_dec done, 3 backward_dec done
  int live = 0; size_t peak_bytes = 0;
};
