#include <algorithm>
// exec.cu - pulse_stage_forward / pulse_stage_backward / temb and loss helpers:
// walks the op plan and enqueues kernels.  Rows a1-a11 of SURVEY.md 8a.
#include "stage.h"
#include "toggles.h"

#include <cstdlib>
#include <cstring>

using namespace pulse;

namespace {

struct Ctx {
  pulse_stage* s;
  char* skip;     // base of this microbatch's skip-cache slot
  char* stash;    // base of this microbatch's stash
  char* work;     // per-stage workspace
  cudaStream_t st;
  cudaStream_t side = nullptr;   // non-null: kernels off the critical chain go here (weight gradients, shortcut convs ...)
  cudaStream_t side2 = nullptr;  // non-null (with side): the tail of the backward runs here, beside both
  int ev_proj = -1;              // forward: side-stream event after the temb projections
  int n_ev = 0;                  // events of s->sync_events used by this call
  int rb_count = 0;              // ResBlocks processed so far in this backward (g_h1 double buffer / hazard events)
  int ev_rb[2] = {-1, -1};       // event recorded on the side stream after the wgrads of the last ResBlock of each parity
  int dt;
  // backward: what the tail (bias / temb-projection gradients of every op, then optionally the timestep-MLP
  // backward) needs; it is enqueued beside the chain as soon as the last g_p is complete (tail_work)
  const float* emb = nullptr; float* g_temb = nullptr; const float* temb_stash = nullptr;
  int acc_w = 0, acc_temb = 0; bool last_op = false, tail_done = false;
  bool own_ok = true;      // this call also zeroes the gradient buffer (not the encoder half of a split stage): see run_wgrad
  int op_lo = 0, op_hi = 0;      // ops this call runs: [op_lo, op_hi)
  bool err = false;
  cudaEvent_t new_event() {
    if (n_ev == (int)s->sync_events.size()) {
      cudaEvent_t e;
      cudaEventCreateWithFlags(&e, cudaEventDisableTiming);
      s->sync_events.push_back(e);
    }
    return s->sync_events[n_ev++];
  }
  // side stream continues after everything enqueued on the main stream so far
  void fork() {
    if (!side) return;
    cudaEvent_t e = new_event();
    cudaEventRecord(e, st);
    cudaStreamWaitEvent(side, e, 0);
  }
  int mark_side() {              // returns the index of an event recorded on the side stream now
    cudaEvent_t e = new_event();
    cudaEventRecord(e, side);
    return n_ev - 1;
  }
  void wait_side(int ev) { if (side && ev >= 0) cudaStreamWaitEvent(st, s->sync_events[ev], 0); }
  bool in_rb = false;
  cudaStream_t wst() const { return side ? side : st; }      // weight gradients: beside the chain when there is a side stream
  // boundary tensors that nothing reads after this call live directly in the caller's buffers (no copy):
  // d_out (forward), g_d_out / g_h_in / g_x_in (backward)
  int ov_ft = -1; char* ov_fp = nullptr;
  int ov_gt[3] = {-1, -1, -1}; char* ov_gp[3] = {nullptr, nullptr, nullptr};
  char* fwd(int t) const {
    if (t == ov_ft) return ov_fp;
    const TRef& r = s->tensors[t].ref;
    return (r.region == R_SKIP ? skip : r.region == R_STASH ? stash : work) + r.off;
  }
  char* grad(int t) const {
    for (int i = 0; i < 3; ++i) if (t == ov_gt[i]) return ov_gp[i];
    return (s->tensors[t].g_in_stash ? stash : work) + s->tensors[t].goff;
  }
  const char* par(int p) const { return s->d_params + s->params[p].off; }
  float* pgrad(int p) const { return (float*)((char*)s->d_grads + s->params[p].goff); }
  size_t bytes(int t) const {
    const TRef& r = s->tensors[t].ref;
    return (size_t)s->d.n * r.h * r.w * r.c * s->esz();
  }
  bool tc() const { return dt == DT_BF16 && !(s->d.flags & PULSE_FLAG_FORCE_SIMT); }
};

// launches inside the scope go to the side stream (if there is one)
struct OnSide {
  Ctx& c; cudaStream_t saved;
  explicit OnSide(Ctx& c_) : c(c_), saved(c_.st) { if (c.side) c.st = c.side; }
  ~OnSide() { c.st = saved; }
};
void setup_side(pulse_stage* s, Ctx& c) {
  if (s->side_mode < 0) s->side_mode = toggles().no_side_stream ? 0 : 1;
  if (s->side_mode == 1 && !s->profiling) {
    if (!s->side && cudaStreamCreateWithFlags(&s->side, cudaStreamNonBlocking) != cudaSuccess) { s->side = nullptr; return; }
    c.side = s->side;
    if (!s->side2 && cudaStreamCreateWithFlags(&s->side2, cudaStreamNonBlocking) != cudaSuccess) s->side2 = nullptr;
    c.side2 = s->side2;
  }
}


// profiling span around a group of launches of one kernel class
struct Prof {
  pulse_stage* s; cudaStream_t st; int idx = -1; uint64_t l0;
  Prof(pulse_stage* s_, cudaStream_t st_, int klass, double flops, double bytes) : s(s_), st(st_), l0(s_->launches) {
    if (!s->profiling) return;
    cudaEvent_t ev[2];
    for (int i = 0; i < 2; ++i) {
      if (!s->event_pool.empty()) { ev[i] = s->event_pool.back(); s->event_pool.pop_back(); }
      else if (cudaEventCreate(&ev[i]) != cudaSuccess) return;
    }
    cudaEventRecord(ev[0], st);
    s->spans.push_back({klass, ev[0], ev[1], flops, bytes, 0});
    idx = (int)s->spans.size() - 1;
  }
  ~Prof() {
    if (idx < 0) return;
    cudaEventRecord(s->spans[idx].e1, st);
    s->spans[idx].launches = (int)(s->launches - l0);
  }
};

double conv_flops(const ConvArgs& a) {      // EXECUTED flops
  if (a.mode == CONV_UP2) return 2.0 * a.n * a.hin * a.win * a.cout * a.src.c() * 16;          // 4 phases x 4 taps on the low-res grid
  if (a.mode == CONV_UP2_DGRAD) return 2.0 * a.n * a.hout * a.wout * a.cout * a.src.c() * 16;
  const double mpix = a.mode == CONV_DGRAD_S2 ? (double)a.n * a.hin * a.win : (double)a.n * a.hout * a.wout;
  return 2.0 * mpix * a.cout * a.src.c() * a.ksize * a.ksize;     // the s2 dgrad phases execute exactly 9/4 taps per output
}
void run_stats(Ctx& c, int t);
void tail_work(Ctx& c);
// stats_t >= 0: the conv writes tensor stats_t, which a GroupNorm will read: its channel stats come from the conv
// epilogue where the kernel supports it, else from a chan_stats pass
void run_conv(Ctx& c, ConvArgs a, int stats_t = -1) {
  const bool tc = c.tc() && conv_tc_any_supported(a);
  bool fused = false;
  if (stats_t >= 0 && c.s->tensors[stats_t].gn_input) {
    a.cst = (float*)(c.stash + c.s->tensors[stats_t].cst);
    fused = tc && conv_emits_stats(a);
    if (!fused) a.cst = nullptr;
  }
  {
    Prof pr(c.s, c.st, tc ? PULSE_KCLASS_CONV_TC : PULSE_KCLASS_CONV_SIMT, conv_flops(a), 0.0);
    const int r = tc ? conv_tc_any(a, c.st) : conv_simt(a, c.st);
    if (r < 0) c.err = true; else c.s->launches += r;
  }
  if (stats_t >= 0 && !fused) run_stats(c, stats_t);
}
void run_wgrad(Ctx& c, const WgradArgs& a) {
  const bool tc = c.tc() && wgrad_tc_any_supported(a);
  Prof pr(c.s, c.wst(), tc ? PULSE_KCLASS_WGRAD_TC : PULSE_KCLASS_CONV_SIMT,
          a.up2 ? 2.0 * a.n * a.hin * a.win * a.cout * a.src.c() * 16
                : 2.0 * a.n * a.hout * a.wout * a.cout * a.src.c() * a.ksize * a.ksize, 0.0);
  WgradArgs b = a;
  if (tc && c.own_ok && wgrad_whole_tiles(a)) {
    const size_t off = (size_t)((const char*)a.dw - (const char*)c.s->d_grads);
    if (c.s->own_valid) b.overwrite = !c.acc_w;       // (its range was left out of the zeroing: backward_impl)
    else c.s->own_runs.push_back({off, (size_t)a.cout * a.ksize * a.ksize * a.src.c() * sizeof(float)});
  }
  const int r = tc ? wgrad_tc_any(b, c.wst()) : wgrad_simt(b, c.wst());
  if (r < 0) c.err = true; else c.s->launches += r;
}
// GroupNorm+SiLU wrappers: algorithmic bytes 2 x esz per element forward, 3 x esz backward
float* cst_of(const Ctx& c, int t) { return t < 0 ? nullptr : (float*)(c.stash + c.s->tensors[t].cst); }
float* cs_of(const Ctx& c, int t) {      // fused pixel sums of the gradient of tensor t, if its writers emit them
  const Tensor& T = c.s->tensors[t];
  return (T.is_out && T.cs_fused) ? (float*)(c.work + T.cs) : nullptr;
}
// channel stats of a freshly written tensor that a GroupNorm will read
void run_stats(Ctx& c, int t) {
  pulse_stage* s = c.s;
  const Tensor& T = s->tensors[t];
  if (!T.gn_input) return;
  const int hw = T.ref.h * T.ref.w;
  Prof pr(s, c.st, PULSE_KCLASS_GN_FWD, 0.0, 0.0);      // its bytes are not algorithmic: counted as GroupNorm-forward time
  s->launches += chan_stats(c.dt, c.fwd(t), s->d.n, hw, T.ref.c, cst_of(c, t), c.st);
}
void run_gn_fwd(Ctx& c, Cat x, int t0, int t1, int hw, const void* gamma, const void* beta, size_t mr, void* a_out,
                int act = 1) {
  pulse_stage* s = c.s;
  Prof pr(s, c.st, PULSE_KCLASS_GN_FWD, 0.0, 2.0 * s->esz() * s->d.n * hw * x.c());
  s->launches += gn_silu_fwd(c.dt, x, s->d.n, hw, s->d.groups, s->d.eps, gamma, beta, cst_of(c, t0), cst_of(c, t1),
                             (float*)(c.stash + mr), a_out, c.st, act);
}
void run_gn_bwd(Ctx& c, const void* g_a, Cat x, size_t mr, int hw, const void* gamma, const void* beta,
                size_t bst, const void* add, void* dst0, int dc0, int acc0, void* dst1, int acc1, float* dgamma,
                float* dbeta, float* cs0, float* cs1, int act = 1) {
  pulse_stage* s = c.s;
  Prof pr(s, c.st, PULSE_KCLASS_GN_BWD, 0.0, (3.0 + (add ? 1.0 : 0.0)) * s->esz() * s->d.n * hw * x.c());
  s->launches += gn_silu_bwd(c.dt, g_a, x, s->d.n, hw, s->d.groups, s->d.eps, gamma, beta,
                             (const float*)(c.stash + mr), (float*)(c.work + bst), add, dst0, dc0, acc0, dst1, acc1, dgamma, dbeta,
                             cs0, cs1, c.st, !(s->d.flags & PULSE_FLAG_GN_TWO_PASS), true, act);
}

ConvArgs conv_args(const Ctx& c, Cat src, int hin, int win, int hout, int wout, int k, int stride, const void* w,
                   int cout, const void* bias, const float* pn, const void* res, void* out) {
  ConvArgs a;
  a.dt = c.dt; a.src = src; a.n = c.s->d.n; a.hin = hin; a.win = win; a.hout = hout; a.wout = wout;
  a.ksize = k; a.stride = stride; a.mode = CONV_FPROP; a.w = w; a.cout = cout; a.bias = bias; a.pn = pn;
  a.residual = res; a.out = out; a.accumulate = 0;
  a.kernel = (c.s->d.flags & PULSE_FLAG_CONV_PAIR) ? CONV_K_PAIR : (c.s->d.flags & PULSE_FLAG_CONV_1CTA) ? CONV_K_1CTA : CONV_K_AUTO;
  return a;
}

// dgrad of a conv == fprop with the flipped/transposed weights `wt`, which
// prepare_weights() keeps in the workspace
void run_dgrad(Ctx& c, const void* g, int h, int w, int cout, size_t wt_off, int k, int cin, void* g_in,
               int accumulate, int stride, int hin, int win) {
  Cat src{g, cout, nullptr, 0};
  ConvArgs a = conv_args(c, src, h, w, hin, win, k, 1, c.work + wt_off, cin, nullptr, nullptr, nullptr, g_in);
  a.accumulate = accumulate;
  if (stride == 2) a.mode = CONV_DGRAD_S2;
  run_conv(c, a);
}

// ---- nearest-2x upsample + conv as four 2x2 phase convs on the low-resolution tensor (kernels.h CONV_UP2): no upsampled
// tensor, no gradient of it, 4/9 of the FLOPs.  Taken where the tcgen05 kernels cover all three convs of the op; the
// CUDA-core path (fp32, PULSE_FLAG_FORCE_SIMT) keeps the materialised form, which is the oracle's.
ConvArgs up2_fwd_args(const Ctx& c, const OpPlan& op) {
  ConvArgs a = conv_args(c, Cat{c.fwd(op.x0), op.cin, nullptr, 0}, op.hin, op.win, op.hout, op.wout, 3, 1, c.work + op.wt2,
                         op.cout, c.par(op.p[P_C1B]), nullptr, nullptr, c.fwd(op.out));
  a.mode = CONV_UP2;
  return a;
}
ConvArgs up2_dgrad_args(const Ctx& c, const OpPlan& op, const void* g_out) {
  ConvArgs a = conv_args(c, Cat{g_out, op.cout, nullptr, 0}, op.hout, op.wout, op.hin, op.win, 3, 1, c.work + op.wt1, op.cin,
                         nullptr, nullptr, nullptr, c.grad(op.x0));
  a.mode = CONV_UP2_DGRAD;
  return a;
}
WgradArgs up2_wgrad_args(const Ctx& c, const OpPlan& op, const void* g_out) {
  WgradArgs w{c.dt, Cat{c.fwd(op.x0), op.cin, nullptr, 0}, c.s->d.n, op.hin, op.win, g_out, op.hout, op.wout, op.cout, 3, 1,
              c.pgrad(op.p[P_C1W])};
  w.up2 = 1;
  return w;
}
// Which form each of the three convs of an up op takes (include/pulse.h, PULSE_FLAG_UP_*): the weight gradient takes the
// phase form by default (4/9 of the work, exact); the forward and the adjoint need pre-summed bf16 weights (one extra
// weight rounding) and are opt-in.  The 16-tap adjoint has a quarter of the materialised adjoint's tiles with 16/9 of its K:
// it gains only when that adjoint needs more than one wave of tiles; on the few-tile grids of the deep levels the 9-tap
// adjoint on the upsampled grid + 2x2 sum stays even when the flag is set.
int sm_count_cached() {
  static int v = 0;
  if (!v) {
    int dev = 0;
    cudaGetDevice(&dev);
    if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v <= 0) v = 148;
  }
  return v;
}
bool up2_wg(const Ctx& c, const OpPlan& op) {
  return op.kind == PULSE_OP_UP && c.tc() && !(c.s->d.flags & PULSE_FLAG_UP_MATERIALISED) &&
         wgrad_tc_any_supported(up2_wgrad_args(c, op, nullptr));
}
bool up2_fwd(const Ctx& c, const OpPlan& op) {      // only with the phase-form weight gradient: nothing then needs u
  return (c.s->d.flags & PULSE_FLAG_UP_PHASE_FWD) && up2_wg(c, op) && conv_tc_any_supported(up2_fwd_args(c, op));
}
bool up2_dg(const Ctx& c, const OpPlan& op) {
  if (!(c.s->d.flags & PULSE_FLAG_UP_PHASE_DGRAD) || (c.s->d.flags & PULSE_FLAG_UP_MATERIALISED)) return false;
  if (op.kind != PULSE_OP_UP || !c.tc() || !conv_tc_any_supported(up2_dgrad_args(c, op, nullptr))) return false;
  const long long tiles_hi = ((long long)c.s->d.n * op.hout * op.wout + 127) / 128 * (op.cin / (op.cin % 160 == 0 ? 160 : 128));
  return tiles_hi > sm_count_cached();
}

// Wt[ci][k-1-r][k-1-s][co] = W[co][r][s][ci] for the convs of ops [lo, hi), one batched launch.  Redone by the first
// backward after a forward that followed a backward (a new step: parameters may have changed), reused by the other
// backwards of a wave (R21).
void prepare_weights(Ctx& c, int lo, int hi) {
  pulse_stage* s = c.s;
  std::vector<TransposeEntry> e;
  for (int oi = hi - 1; oi >= lo; --oi) {            // in the order the backward needs them
    const OpPlan& op = s->ops[oi];
    const int ctot = op.cin + op.cskip;
    if (op.kind == PULSE_OP_RESBLOCK) {
      e.push_back({c.par(op.p[P_C1W]), c.work + op.wt1, op.cout, 3, ctot});
      e.push_back({c.par(op.p[P_C2W]), c.work + op.wt2, op.cout, 3, op.cout});
      if (op.p[P_SCW] >= 0) e.push_back({c.par(op.p[P_SCW]), c.work + op.wtsc, op.cout, 1, ctot});
    } else if (op.kind == PULSE_OP_TBLOCK) {
      e.push_back({c.par(op.p[P_F2W]), c.work + op.wt4, op.cin, 1, 4 * op.cin});
      e.push_back({c.par(op.p[P_TW]), c.work + op.wt3, 4 * op.cin, 1, op.cin});
      e.push_back({c.par(op.p[P_C2W]), c.work + op.wt2, op.cin, 1, op.cin});
      e.push_back({c.par(op.p[P_C1W]), c.work + op.wt1, 3 * op.cin, 1, op.cin});
      if (op.x1 >= 0) e.push_back({c.par(op.p[P_SCW]), c.work + op.wtsc, op.cin, 1, ctot});
    } else if (op.kind == PULSE_OP_ATTN) {
      e.push_back({c.par(op.p[P_C1W]), c.work + op.wt1, 3 * op.cin, 1, op.cin});
      e.push_back({c.par(op.p[P_C2W]), c.work + op.wt2, op.cin, 1, op.cin});
    } else if (up2_dg(c, op)) {       // WpT [cin][16][cout] for the 16-tap adjoint
      Prof pr(s, c.st, PULSE_KCLASS_OTHER, 0.0, 0.0);
      s->launches += up2_weights(c.dt, c.par(op.p[P_C1W]), op.cout, op.cin, nullptr, c.work + op.wt1, c.st);
    } else {
      e.push_back({c.par(op.p[P_C1W]), c.work + op.wt1, op.cout, 3, op.cin});
    }
  }
  if (e.empty()) return;
  Prof pr(s, c.st, PULSE_KCLASS_OTHER, 0.0, 0.0);
  s->launches += flip_transpose_batch(c.dt, e.data(), (int)e.size(), c.st);
}

void resblock_forward(Ctx& c, const OpPlan& op) {
  pulse_stage* s = c.s;
  const int hw = op.hin * op.win, ctot = op.cin + op.cskip;
  Cat x{c.fwd(op.x0), op.cin, op.x1 >= 0 ? c.fwd(op.x1) : nullptr, op.cskip};
  float* pn = (float*)(c.stash + op.pn);
  // the 1x1 shortcut needs only x: it runs beside the GN1 -> conv1 -> GN2 chain and is joined before conv2
  const void* res = c.fwd(op.x0);
  int ev_sc = -1;
  if (op.p[P_SCW] >= 0) {
    c.fork();
    {
      OnSide g(c);
      run_conv(c, conv_args(c, x, op.hin, op.win, op.hin, op.win, 1, 1, c.par(op.p[P_SCW]), op.cout,
                            c.par(op.p[P_SCB]), nullptr, nullptr, c.fwd(op.out)));
    }
    if (c.side) ev_sc = c.mark_side();
    res = c.fwd(op.out);
  }
  run_gn_fwd(c, x, op.x0, op.x1, hw, c.par(op.p[P_GN1G]), c.par(op.p[P_GN1B]), op.mr1, c.fwd(op.a1));
  if (c.ev_proj >= 0) { c.wait_side(c.ev_proj); c.ev_proj = -1; }      // temb projections (side stream) are ready
  Cat a1{c.fwd(op.a1), ctot, nullptr, 0};
  run_conv(c, conv_args(c, a1, op.hin, op.win, op.hin, op.win, 3, 1, c.par(op.p[P_C1W]), op.cout,
                        c.par(op.p[P_C1B]), pn, nullptr, c.fwd(op.h1)), op.h1);
  Cat h1{c.fwd(op.h1), op.cout, nullptr, 0};
  run_gn_fwd(c, h1, op.h1, -1, hw, c.par(op.p[P_GN2G]), c.par(op.p[P_GN2B]), op.mr2, c.fwd(op.a2));
  c.wait_side(ev_sc);
  Cat a2{c.fwd(op.a2), op.cout, nullptr, 0};
  run_conv(c, conv_args(c, a2, op.hin, op.win, op.hin, op.win, 3, 1, c.par(op.p[P_C2W]), op.cout,
                        c.par(op.p[P_C2B]), nullptr, res, c.fwd(op.out)), op.out);
}

// Self-attention block: xn = GN(x); qkv = conv1x1(xn); o = attention(qkv); out = conv1x1(o) + x
void attn_forward(Ctx& c, const OpPlan& op) {
  pulse_stage* s = c.s;
  const int hw = op.hin * op.win, C = op.cin;
  run_gn_fwd(c, Cat{c.fwd(op.x0), C, nullptr, 0}, op.x0, -1, hw, c.par(op.p[P_GN1G]), c.par(op.p[P_GN1B]), op.mr1,
             c.fwd(op.a1), /*act=*/0);
  run_conv(c, conv_args(c, Cat{c.fwd(op.a1), C, nullptr, 0}, op.hin, op.win, op.hin, op.win, 1, 1, c.par(op.p[P_C1W]), 3 * C,
                        c.par(op.p[P_C1B]), nullptr, nullptr, c.fwd(op.h1)));
  {
    Prof pr(s, c.st, PULSE_KCLASS_OTHER, 4.0 * s->d.n * (double)hw * hw * C, 0.0);
    const int r = attn_fwd(c.dt, c.fwd(op.h1), s->d.n, hw, C, op.heads, c.fwd(op.a2), (float*)(c.stash + op.lse), c.st, c.tc());
    if (r < 0) c.err = true; else s->launches += r;
  }
  run_conv(c, conv_args(c, Cat{c.fwd(op.a2), C, nullptr, 0}, op.hin, op.win, op.hin, op.win, 1, 1, c.par(op.p[P_C2W]), C,
                        c.par(op.p[P_C2B]), nullptr, c.fwd(op.x0), c.fwd(op.out)), op.out);
}

// Transformer block with an optional long skip: see stage.cu for the tensor names
void conv1x1(Ctx& c, Cat src, int h, int w, const void* wgt, int cout, const void* bias, const void* res, void* out) {
  run_conv(c, conv_args(c, src, h, w, h, w, 1, 1, wgt, cout, bias, nullptr, res, out));
}
void tblock_forward(Ctx& c, const OpPlan& op) {
  pulse_stage* s = c.s;
  const int hw = op.hin * op.win, C = op.cin, n = s->d.n;
  const size_t tokens = (size_t)n * hw;
  const char* xs = c.fwd(op.x0);
  if (op.x1 >= 0) {          // the long skip: Linear on the virtual concat [x | skip]
    conv1x1(c, Cat{c.fwd(op.x0), C, c.fwd(op.x1), op.cskip}, op.hin, op.win, c.par(op.p[P_SCW]), C, c.par(op.p[P_SCB]), nullptr,
            c.fwd(op.u));
    xs = c.fwd(op.u);
  }
  s->launches += layernorm_fwd(c.dt, xs, tokens, C, s->d.eps, c.par(op.p[P_GN1G]), c.par(op.p[P_GN1B]),
                               (float*)(c.stash + op.ln1), c.fwd(op.a1), c.st);
  conv1x1(c, Cat{c.fwd(op.a1), C, nullptr, 0}, op.hin, op.win, c.par(op.p[P_C1W]), 3 * C, c.par(op.p[P_C1B]), nullptr, c.fwd(op.h1));
  {
    Prof pr(s, c.st, PULSE_KCLASS_OTHER, 4.0 * n * (double)hw * hw * C, 0.0);
    const int r = attn_fwd(c.dt, c.fwd(op.h1), n, hw, C, op.heads, c.fwd(op.a2), (float*)(c.stash + op.lse), c.st, c.tc());
    if (r < 0) c.err = true; else s->launches += r;
  }
  conv1x1(c, Cat{c.fwd(op.a2), C, nullptr, 0}, op.hin, op.win, c.par(op.p[P_C2W]), C, c.par(op.p[P_C2B]), xs, c.fwd(op.tx1));
  s->launches += layernorm_fwd(c.dt, c.fwd(op.tx1), tokens, C, s->d.eps, c.par(op.p[P_GN2G]), c.par(op.p[P_GN2B]),
                               (float*)(c.stash + op.ln2), c.fwd(op.tl2), c.st);
  conv1x1(c, Cat{c.fwd(op.tl2), C, nullptr, 0}, op.hin, op.win, c.par(op.p[P_TW]), 4 * C, c.par(op.p[P_TB]), nullptr, c.fwd(op.tf1));
  s->launches += gelu_fwd(c.dt, c.fwd(op.tf1), c.fwd(op.tg), tokens * 4 * C, c.st);
  // a GroupNorm never reads a transformer block's output (stats_t = -1 unless a later ResBlock / attention block does)
  run_conv(c, conv_args(c, Cat{c.fwd(op.tg), 4 * C, nullptr, 0}, op.hin, op.win, op.hin, op.win, 1, 1, c.par(op.p[P_F2W]), C,
                        c.par(op.p[P_F2B]), nullptr, c.fwd(op.tx1), c.fwd(op.out)), op.out);
}

// pixel sums of the gradient of an op's output, for its bias gradient: fused by the writers or one colsum pass
void ensure_colsum(Ctx& c, int t) {
  pulse_stage* s = c.s;
  const Tensor& T = s->tensors[t];
  if (T.cs_fused) return;
  Prof pr(s, c.st, PULSE_KCLASS_OTHER, 0.0, 0.0);
  s->launches += colsum(c.dt, c.grad(t), s->d.n, T.ref.h * T.ref.w, T.ref.c, (float*)(c.work + T.cs), c.st);
}

void resblock_backward(Ctx& c, const OpPlan& op) {
  pulse_stage* s = c.s;
  const int n = s->d.n, hw = op.hin * op.win, ctot = op.cin + op.cskip;
  Cat x{c.fwd(op.x0), op.cin, op.x1 >= 0 ? c.fwd(op.x1) : nullptr, op.cskip};
  const int par = c.rb_count & 1;
  c.in_rb = true;
  char* g_out = c.grad(op.out);
  char* g_a2 = c.work + s->w_ga2;
  char* g_h1 = c.work + (par ? s->w_gh1b : s->w_gh1);     // double-buffered: the side stream's wgrad1 reads it late
  char* g_a1 = c.work + s->w_ga1;
  char* g_sc = c.work + s->w_gsc;
  ensure_colsum(c, op.out);
  // conv2 (and shortcut) weight gradients need only g_out: fork them off now
  c.fork();
  int ev_sc = -1;
  if (op.p[P_SCW] >= 0 && c.side) {     // shortcut dgrad needs only g_out: side stream, joined before the GN1 backward
    {
      OnSide g(c);
      run_dgrad(c, g_out, op.hin, op.win, op.cout, op.wtsc, 1, ctot, g_sc, 0, 1, op.hin, op.win);
    }
    ev_sc = c.mark_side();
  }
  WgradArgs w2{c.dt, Cat{c.fwd(op.a2), op.cout, nullptr, 0}, n, op.hin, op.win, g_out, op.hin, op.win, op.cout, 3, 1,
               c.pgrad(op.p[P_C2W])};
  run_wgrad(c, w2);
  if (op.p[P_SCW] >= 0) {
    WgradArgs ws{c.dt, x, n, op.hin, op.win, g_out, op.hin, op.win, op.cout, 1, 1, c.pgrad(op.p[P_SCW])};
    run_wgrad(c, ws);
  }
  run_dgrad(c, g_out, op.hin, op.win, op.cout, op.wt2, 3, op.cout, g_a2, 0, 1, op.hin, op.win);
  // GN2 + SiLU backward -> g_h1, and its pixel sums g_p[n,c] (temb projection / conv1 bias gradients).
  // g_h1 of this parity was last read by the wgrad1 of the ResBlock two back: wait for it.
  c.wait_side(c.ev_rb[par]);
  run_gn_bwd(c, g_a2, Cat{c.fwd(op.h1), op.cout, nullptr, 0}, op.mr2, hw, c.par(op.p[P_GN2G]), c.par(op.p[P_GN2B]),
             op.bst2, nullptr, g_h1, op.cout, 0, nullptr, 0, c.pgrad(op.p[P_GN2G]), c.pgrad(op.p[P_GN2B]),
             (float*)(c.work + op.gp), nullptr);
  // conv1: wgrad (side stream), dgrad
  c.fork();
  if (c.last_op && c.side2) tail_work(c);      // every g_p is complete: the tail runs beside conv1 / GN1 of this block
  WgradArgs w1{c.dt, Cat{c.fwd(op.a1), ctot, nullptr, 0}, n, op.hin, op.win, g_h1, op.hin, op.win, op.cout, 3, 1,
               c.pgrad(op.p[P_C1W])};
  run_wgrad(c, w1);
  if (c.side) c.ev_rb[par] = c.mark_side();
  run_dgrad(c, g_h1, op.hin, op.win, op.cout, op.wt1, 3, ctot, g_a1, 0, 1, op.hin, op.win);
  // shortcut
  const void* add = g_out;
  if (op.p[P_SCW] >= 0) {
    if (c.side) c.wait_side(ev_sc);
    else run_dgrad(c, g_out, op.hin, op.win, op.cout, op.wtsc, 1, ctot, g_sc, 0, 1, op.hin, op.win);
    add = g_sc;
  }
  // GN1 + SiLU backward, split into g_h and g_skip (skip gradient accumulated locally)
  run_gn_bwd(c, g_a1, x, op.mr1, hw, c.par(op.p[P_GN1G]), c.par(op.p[P_GN1B]), op.bst1, add, c.grad(op.x0), op.cin,
             op.acc_x0, op.x1 >= 0 ? c.grad(op.x1) : nullptr, op.acc_x1, c.pgrad(op.p[P_GN1G]), c.pgrad(op.p[P_GN1B]),
             cs_of(c, op.x0), op.x1 >= 0 ? cs_of(c, op.x1) : nullptr);
  ++c.rb_count;
  c.in_rb = false;
}

void attn_backward(Ctx& c, const OpPlan& op) {
  pulse_stage* s = c.s;
  const int n = s->d.n, hw = op.hin * op.win, C = op.cin;
  char* g_out = c.grad(op.out);
  char* g_o = c.work + s->w_ga2;
  char* g_qkv = c.work + s->w_gqkv;
  char* g_xn = c.work + s->w_ga1;
  ensure_colsum(c, op.out);
  c.fork();
  run_wgrad(c, WgradArgs{c.dt, Cat{c.fwd(op.a2), C, nullptr, 0}, n, op.hin, op.win, g_out, op.hin, op.win, C, 1, 1,
                         c.pgrad(op.p[P_C2W])});
  run_dgrad(c, g_out, op.hin, op.win, C, op.wt2, 1, C, g_o, 0, 1, op.hin, op.win);
  {
    Prof pr(s, c.st, PULSE_KCLASS_OTHER, 10.0 * n * (double)hw * hw * C, 0.0);
    const int r = attn_bwd(c.dt, c.fwd(op.h1), g_o, n, hw, C, op.heads, (float*)(c.stash + op.lse), g_qkv, c.st, c.tc());
    if (r < 0) c.err = true; else s->launches += r;
    s->launches += colsum(c.dt, g_qkv, n, hw, 3 * C, (float*)(c.work + op.gp), c.st);      // qkv bias gradient
  }
  c.fork();
  if (c.last_op && c.side2) tail_work(c);
  run_wgrad(c, WgradArgs{c.dt, Cat{c.fwd(op.a1), C, nullptr, 0}, n, op.hin, op.win, g_qkv, op.hin, op.win, 3 * C, 1, 1,
                         c.pgrad(op.p[P_C1W])});
  // the side stream's wgrad reads g_qkv: the next attention block's backward must not overwrite it before that (one
  // shared buffer): join here
  if (c.side) c.wait_side(c.mark_side());
  run_dgrad(c, g_qkv, op.hin, op.win, 3 * C, op.wt1, 1, C, g_xn, 0, 1, op.hin, op.win);
  run_gn_bwd(c, g_xn, Cat{c.fwd(op.x0), C, nullptr, 0}, op.mr1, hw, c.par(op.p[P_GN1G]), c.par(op.p[P_GN1B]), op.bst1,
             g_out, c.grad(op.x0), C, op.acc_x0, nullptr, 0, c.pgrad(op.p[P_GN1G]), c.pgrad(op.p[P_GN1B]), cs_of(c, op.x0),
             nullptr, /*act=*/0);
}

void tblock_backward(Ctx& c, const OpPlan& op) {
  pulse_stage* s = c.s;
  const int n = s->d.n, hw = op.hin * op.win, C = op.cin, H = op.hin, Wd = op.win, ctot = C + op.cskip;
  const size_t tokens = (size_t)n * hw;
  const bool skip = op.x1 >= 0;
  const char* xs = skip ? c.fwd(op.u) : c.fwd(op.x0);
  char* g_out = c.grad(op.out);
  char* g_g = c.work + s->w_t4a;  char* g_f1 = c.work + s->w_t4b;
  char* g_l2 = c.work + s->w_tca; char* g_x1 = c.work + s->w_tcb;
  char* g_o = c.work + s->w_tca;  char* g_l1 = c.work + s->w_tca;      // g_l2, g_o, g_l1 are never live together
  char* g_qkv = c.work + s->w_gqkv; char* g_xs = c.work + s->w_ga1;
  float* gp = (float*)(c.work + op.gp);                                // [n][c] | [n][3c] | [n][c] | [n][4c]
  float* gp_xs = gp; float* gp_qkv = gp + (size_t)n * C; float* gp_x1 = gp + (size_t)n * 4 * C; float* gp_f1 = gp + (size_t)n * 5 * C;
  auto wg = [&](const void* src, int cs, const void* src1, int cs1, const void* g, int cout, int pidx) {
    run_wgrad(c, WgradArgs{c.dt, Cat{src, cs, src1, cs1}, n, H, Wd, g, H, Wd, cout, 1, 1, c.pgrad(op.p[pidx])});
  };
  ensure_colsum(c, op.out);                                            // fc2 bias
  c.fork();
  wg(c.fwd(op.tg), 4 * C, nullptr, 0, g_out, C, P_F2W);
  run_dgrad(c, g_out, H, Wd, C, op.wt4, 1, 4 * C, g_g, 0, 1, H, Wd);
  s->launches += gelu_bwd(c.dt, c.fwd(op.tf1), g_g, g_f1, tokens * 4 * C, c.st);
  s->launches += colsum(c.dt, g_f1, n, hw, 4 * C, gp_f1, c.st);       // fc1 bias
  c.fork();
  wg(c.fwd(op.tl2), C, nullptr, 0, g_f1, 4 * C, P_TW);
  run_dgrad(c, g_f1, H, Wd, 4 * C, op.wt3, 1, C, g_l2, 0, 1, H, Wd);
  // g_x1 = LN2'(g_l2) + g_out
  s->launches += layernorm_bwd(c.dt, g_l2, c.fwd(op.tx1), tokens, C, c.par(op.p[P_GN2G]), (const float*)(c.stash + op.ln2), g_out,
                               g_x1, 0, c.pgrad(op.p[P_GN2G]), c.pgrad(op.p[P_GN2B]), c.st);
  s->launches += colsum(c.dt, g_x1, n, hw, C, gp_x1, c.st);           // proj bias
  c.fork();
  wg(c.fwd(op.a2), C, nullptr, 0, g_x1, C, P_C2W);
  run_dgrad(c, g_x1, H, Wd, C, op.wt2, 1, C, g_o, 0, 1, H, Wd);
  {
    Prof pr(s, c.st, PULSE_KCLASS_OTHER, 10.0 * n * (double)hw * hw * C, 0.0);
    const int r = attn_bwd(c.dt, c.fwd(op.h1), g_o, n, hw, C, op.heads, (float*)(c.stash + op.lse), g_qkv, c.st, c.tc());
    if (r < 0) c.err = true; else s->launches += r;
    s->launches += colsum(c.dt, g_qkv, n, hw, 3 * C, gp_qkv, c.st);   // qkv bias
  }
  c.fork();
  wg(c.fwd(op.a1), C, nullptr, 0, g_qkv, 3 * C, P_C1W);
  run_dgrad(c, g_qkv, H, Wd, 3 * C, op.wt1, 1, C, g_l1, 0, 1, H, Wd);
  // g_xs = LN1'(g_l1) + g_x1: the block's input gradient, or (long skip) the gradient of the Linear's output
  if (!skip) {
    s->launches += layernorm_bwd(c.dt, g_l1, xs, tokens, C, c.par(op.p[P_GN1G]), (const float*)(c.stash + op.ln1), g_x1,
                                 c.grad(op.x0), op.acc_x0, c.pgrad(op.p[P_GN1G]), c.pgrad(op.p[P_GN1B]), c.st);
  } else {
    s->launches += layernorm_bwd(c.dt, g_l1, xs, tokens, C, c.par(op.p[P_GN1G]), (const float*)(c.stash + op.ln1), g_x1, g_xs, 0,
                                 c.pgrad(op.p[P_GN1G]), c.pgrad(op.p[P_GN1B]), c.st);
    s->launches += colsum(c.dt, g_xs, n, hw, C, gp_xs, c.st);         // skip Linear bias
    c.fork();
    wg(c.fwd(op.x0), C, c.fwd(op.x1), op.cskip, g_xs, C, P_SCW);
    // the Linear's adjoint, one 1x1 conv per source: rows [0, C) / [C, C + skip) of the transposed weight [C + skip][C]
    const size_t esz = s->esz();
    run_dgrad(c, g_xs, H, Wd, C, op.wtsc, 1, C, c.grad(op.x0), op.acc_x0, 1, H, Wd);
    run_dgrad(c, g_xs, H, Wd, C, op.wtsc + (size_t)C * C * esz, 1, op.cskip, c.grad(op.x1), op.acc_x1, 1, H, Wd);
    (void)ctot;
  }
  // the side stream's weight gradients read the shared gradient buffers of this block: join before the next block reuses them
  if (c.side) c.wait_side(c.mark_side());
  if (c.last_op && c.side2) tail_work(c);
}

// bias / temb-projection gradients of every op from the pixel sums, in one batched launch (row a8-a10)
void small_grads(Ctx& c, const float* emb, float* g_temb, cudaStream_t st) {
  pulse_stage* s = c.s;
  std::vector<SmallGradEntry> e;
  for (int oi = c.op_lo; oi < c.op_hi; ++oi) {       // the ops of this call (all of them, or one half of a split stage)
    const OpPlan& op = s->ops[oi];
    SmallGradEntry g;
    memset(&g, 0, sizeof g);
    g.cs_out = (const float*)(c.work + s->tensors[op.out].cs);
    g.cout = op.cout;
    if (op.kind == PULSE_OP_RESBLOCK) {
      g.db_out = c.pgrad(op.p[P_C2B]);
      g.db_out2 = op.p[P_SCB] >= 0 ? c.pgrad(op.p[P_SCB]) : nullptr;
      g.gp = (const float*)(c.work + op.gp);
      g.db1 = c.pgrad(op.p[P_C1B]); g.dtb = c.pgrad(op.p[P_TB]); g.dtw = c.pgrad(op.p[P_TW]); g.tw = c.par(op.p[P_TW]);
    } else if (op.kind == PULSE_OP_TBLOCK) {
      g.db_out = c.pgrad(op.p[P_F2B]);            // fc2 bias from the pixel sums of g_out
      const float* gp = (const float*)(c.work + op.gp);
      const int C = op.cin, n = s->d.n;
      auto extra = [&](const float* sums, int width, int pidx) {
        SmallGradEntry q;
        memset(&q, 0, sizeof q);
        q.cs_out = sums; q.db_out = c.pgrad(op.p[pidx]); q.cout = width;
        e.push_back(q);
      };
      if (op.x1 >= 0) extra(gp, C, P_SCB);
      extra(gp + (size_t)n * C, 3 * C, P_C1B);
      extra(gp + (size_t)n * 4 * C, C, P_C2B);
      extra(gp + (size_t)n * 5 * C, 4 * C, P_TB);
    } else if (op.kind == PULSE_OP_ATTN) {
      g.db_out = c.pgrad(op.p[P_C2B]);            // proj bias from the pixel sums of g_out
      SmallGradEntry q;                           // qkv bias from the pixel sums of g_qkv
      memset(&q, 0, sizeof q);
      q.cs_out = (const float*)(c.work + op.gp); q.db_out = c.pgrad(op.p[P_C1B]); q.cout = 3 * op.cin;
      e.push_back(q);
    } else {
      g.db_out = c.pgrad(op.p[P_C1B]);
    }
    e.push_back(g);
  }
  if (e.empty()) return;
  Prof pr(s, st, PULSE_KCLASS_OTHER, 0.0, 0.0);
  s->launches += small_grads_batch(c.dt, emb, g_temb, s->d.n, s->d.temb_dim, e.data(), (int)e.size(), st);
}
pulse_status_t temb_backward_impl(pulse_stage* s, const float* d_g_emb, const float* d_stash, int accumulate_wgrad,
                                  cudaStream_t st);
// bias / temb-projection gradients of every op, then (pulse_stage_backward_temb) the timestep-MLP backward; on the
// side stream when there is one (the caller has forked it), so that none of it is left for the end of the step
void tail_work(Ctx& c) {
  cudaStream_t st = c.side2 ? c.side2 : (c.side ? c.side : c.st);
  if (c.side2) {                                   // side2 continues after everything enqueued on the main stream so far
    cudaEvent_t e = c.new_event();
    cudaEventRecord(e, c.st);
    cudaStreamWaitEvent(c.side2, e, 0);
  }
  small_grads(c, c.emb, c.g_temb, st);
  if (c.temb_stash && temb_backward_impl(c.s, c.g_temb, c.temb_stash, c.acc_temb, st) != PULSE_OK) c.err = true;
  c.tail_done = true;
}

pulse_status_t check_bound(pulse_stage* s, pulse_skip_cache* cache) {
  if (!s || !cache) return fail(PULSE_ERR_INVALID_ARG, "null stage / cache");
  if (cache->stage != s) return fail(PULSE_ERR_INVALID_ARG, "cache belongs to another stage");
  if (!s->d_params || !s->d_grads) return fail(PULSE_ERR_STATE, "parameters not bound");
  if (!s->d_work) return fail(PULSE_ERR_STATE, "workspace not bound");
  return PULSE_OK;
}

}  // namespace

namespace {
pulse_status_t temb_forward_impl(pulse_stage* s, const int64_t* d_t, float* d_emb, float* d_stash, cudaStream_t st);
}
enum { PART_ENC = 1, PART_DEC = 2, PART_ALL = 3 };      // halves of a split (pipeline) stage; PART_ALL: the one-call forms

// d_t != nullptr (pulse_stage_forward_temb): the embedding is computed here, beside the stash of the boundary tensors,
// from the timesteps into d_temb (written) with its MLP stash in d_temb_stash
static pulse_status_t forward_impl(pulse_stage_t* s, pulse_skip_cache_t* cache, int64_t mb, const void* d_x_in,
                                   const void* d_h_in, float* d_temb, const int64_t* d_t, float* d_temb_stash,
                                   void* d_e_out, void* d_d_out, void* stream, int parts = PART_ALL) {
  pulse_status_t stt = check_bound(s, cache);
  if (stt) return stt;
  const bool open = s->d.link == PULSE_LINK_OPEN;
  const bool enc = parts & PART_ENC, dec = parts & PART_DEC;
  if (parts != PART_ALL && !(s->d.flags & PULSE_FLAG_SPLIT)) return fail(PULSE_ERR_STATE, "the two-call forms need PULSE_FLAG_SPLIT");
  if (mb < 0) return fail(PULSE_ERR_INVALID_ARG, "negative mb_id");
  if (enc && (!d_x_in || !d_temb)) return fail(PULSE_ERR_INVALID_ARG, "null x_in / temb");
  if (dec && !d_d_out) return fail(PULSE_ERR_INVALID_ARG, "null d_out");
  if (open && ((enc && !d_e_out) || (dec && !d_h_in))) return fail(PULSE_ERR_INVALID_ARG, "OPEN stage needs h_in and e_out");
  if (!open && (d_h_in || d_e_out)) return fail(PULSE_ERR_INVALID_ARG, "CLOSED stage takes no h_in / e_out");
  int slot = -1;
  if (enc) {
    for (int i = 0; i < cache->slots; ++i) {
      if (cache->mb[i] == mb) return fail(PULSE_ERR_CACHE, "microbatch %lld is already live", (long long)mb);
      if (cache->mb[i] < 0 && slot < 0) slot = i;
    }
    if (slot < 0) return fail(PULSE_ERR_CACHE, "skip cache full (%d slots)", cache->slots);
  } else {
    for (int i = 0; i < cache->slots; ++i) if (cache->mb[i] == mb) slot = i;
    if (slot < 0 || cache->phase[slot] != 1)
      return fail(PULSE_ERR_STATE, "forward_dec of microbatch %lld without a forward_enc", (long long)mb);
  }
  Ctx c;
  c.s = s; c.st = (cudaStream_t)stream; c.dt = s->d.dtype == PULSE_F32 ? DT_F32 : DT_BF16;
  c.skip = cache->base + (size_t)slot * cache->bytes_per_slot;
  c.work = s->d_work;
  c.stash = s->d_work + s->work_bytes + (size_t)slot * s->stash_bytes;
  const int n_first = s->n_enc + s->n_mid, nops = (int)s->ops.size();
  c.op_lo = enc ? 0 : n_first; c.op_hi = dec ? nops : n_first;
  float* emb = (float*)(c.stash + s->emb_off);
  if (dec && s->tensors[s->t_dout].ref.region == R_STASH && ((uintptr_t)d_d_out & 255) == 0) { c.ov_ft = s->t_dout; c.ov_fp = (char*)d_d_out; }
  // a boundary tensor that a GroupNorm reads is stashed and measured in one pass (stash_in below); the rest are copies
  const bool fuse_x = s->tensors[s->t_xin].gn_input, fuse_h = open && s->tensors[s->t_hin].gn_input;
  if (enc) {
    // channel stats of every GroupNorm input of the slot, both halves: zeroed once, when the slot is taken
    if (s->cst_end > s->cst_begin) CK_CUDA(cudaMemsetAsync(c.stash + s->cst_begin, 0, s->cst_end - s->cst_begin, c.st));
    if (!fuse_x) CK_CUDA(cudaMemcpyAsync(c.fwd(s->t_xin), d_x_in, c.bytes(s->t_xin), cudaMemcpyDeviceToDevice, c.st));
    if (!d_t) CK_CUDA(cudaMemcpyAsync(emb, d_temb, (size_t)s->d.n * s->d.temb_dim * 4, cudaMemcpyDeviceToDevice, c.st));
  }
  if (dec && open && !fuse_h) CK_CUDA(cudaMemcpyAsync(c.fwd(s->t_hin), d_h_in, c.bytes(s->t_hin), cudaMemcpyDeviceToDevice, c.st));
  setup_side(s, c);
  if (enc) {   // beside the chain (side stream): (one-call form) the timestep MLP, then p[n,c] = Wt SiLU(emb) + bt of every
               // ResBlock of BOTH halves in one launch (row a1), joined before the first conv1
    c.fork();
    OnSide g(c);
    if (d_t) {
      if (temb_forward_impl(s, d_t, d_temb, d_temb_stash, c.st) != PULSE_OK) c.err = true;
      CK_CUDA(cudaMemcpyAsync(emb, d_temb, (size_t)s->d.n * s->d.temb_dim * 4, cudaMemcpyDeviceToDevice, c.st));
    }
    if (s->last_was_backward) s->wp_valid = false;      // a forward after a backward starts a new step: parameters may have changed
    if (!s->wp_valid) {                                  // pre-summed phase weights Wp [4][cout][4][cin] of the up convs
      for (const OpPlan& op : s->ops)
        if (up2_fwd(c, op)) {
          Prof pr(s, c.st, PULSE_KCLASS_OTHER, 0.0, 0.0);
          s->launches += up2_weights(c.dt, c.par(op.p[P_C1W]), op.cout, op.cin, c.work + op.wt2, nullptr, c.st);
        }
      s->wp_valid = true;
    }
    std::vector<ProjEntry> pe;
    for (const OpPlan& op : s->ops)
      if (op.kind == PULSE_OP_RESBLOCK)
        pe.push_back({c.par(op.p[P_TW]), c.par(op.p[P_TB]), (float*)(c.stash + op.pn), op.cout});
    if (!pe.empty()) {
      Prof pr(s, c.st, PULSE_KCLASS_OTHER, 0.0, 0.0);
      s->launches += temb_proj_batch(c.dt, emb, s->d.n, s->d.temb_dim, pe.data(), (int)pe.size(), c.st);
    }
    if (c.side) c.ev_proj = c.mark_side();
  }
  auto stash_in = [&](int t, const void* src) {      // channel stats of `src` + its copy into the stage's tensor t
    const Tensor& T = s->tensors[t];
    Prof pr(s, c.st, PULSE_KCLASS_GN_FWD, 0.0, 0.0);
    s->launches += chan_stats(c.dt, src, s->d.n, T.ref.h * T.ref.w, T.ref.c, cst_of(c, t), c.st, c.fwd(t));
  };
  if (enc && fuse_x) stash_in(s->t_xin, d_x_in);
  if (dec && fuse_h) stash_in(s->t_hin, d_h_in);
  for (int i = c.op_lo; i < c.op_hi; ++i) {
    const OpPlan& op = s->ops[i];
    switch (op.kind) {
      case PULSE_OP_RESBLOCK: resblock_forward(c, op); break;
      case PULSE_OP_ATTN: attn_forward(c, op); break;
      case PULSE_OP_TBLOCK: tblock_forward(c, op); break;
      case PULSE_OP_CONV_IN:
      case PULSE_OP_DOWN: {
        const int stride = op.kind == PULSE_OP_DOWN ? 2 : 1;
        run_conv(c, conv_args(c, Cat{c.fwd(op.x0), op.cin, nullptr, 0}, op.hin, op.win, op.hout, op.wout, 3, stride,
                              c.par(op.p[P_C1W]), op.cout, c.par(op.p[P_C1B]), nullptr, nullptr, c.fwd(op.out)), op.out);
        break;
      }
      case PULSE_OP_UP: {
        if (up2_fwd(c, op)) {
          if (c.ev_proj >= 0) { c.wait_side(c.ev_proj); c.ev_proj = -1; }      // the phase weights (side stream) are ready
          run_conv(c, up2_fwd_args(c, op), op.out);
          break;
        }
        s->launches += upsample2(c.dt, c.fwd(op.x0), s->d.n, op.hin, op.win, op.cin, c.fwd(op.u), c.st);
        run_conv(c, conv_args(c, Cat{c.fwd(op.u), op.cin, nullptr, 0}, op.hout, op.wout, op.hout, op.wout, 3, 1,
                              c.par(op.p[P_C1W]), op.cout, c.par(op.p[P_C1B]), nullptr, nullptr, c.fwd(op.out)), op.out);
        break;
      }
      case PULSE_OP_HEAD: {
        run_gn_fwd(c, Cat{c.fwd(op.x0), op.cin, nullptr, 0}, op.x0, -1, op.hin * op.win, c.par(op.p[P_GN1G]),
                   c.par(op.p[P_GN1B]), op.mr1, c.fwd(op.a1));
        run_conv(c, conv_args(c, Cat{c.fwd(op.a1), op.cin, nullptr, 0}, op.hin, op.win, op.hin, op.win, 3, 1,
                              c.par(op.p[P_C1W]), op.cout, c.par(op.p[P_C1B]), nullptr, nullptr, c.fwd(op.out)));
        break;
      }
    }
  }
  if (c.side) c.wait_side(c.mark_side());       // join
  if (s->last_was_backward) s->wt_valid = false;      // a forward after a backward starts a new step: the parameters may have changed
  s->last_was_backward = false;
  if (enc && open) CK_CUDA(cudaMemcpyAsync(d_e_out, c.fwd(s->t_eout), c.bytes(s->t_eout), cudaMemcpyDeviceToDevice, c.st));
  if (dec && c.ov_ft < 0) CK_CUDA(cudaMemcpyAsync(d_d_out, c.fwd(s->t_dout), c.bytes(s->t_dout), cudaMemcpyDeviceToDevice, c.st));
  if (c.err) return fail(PULSE_ERR_CUDA, "tensor-core conv launch failed: %s", tc_last_error());
  CK_CUDA(cudaGetLastError());
  if (enc) {
    cache->mb[slot] = mb;
    cache->live++;
    const size_t lb = (size_t)cache->live * cache->bytes_per_slot;
    if (lb > cache->peak_bytes) cache->peak_bytes = lb;
  }
  cache->phase[slot] = dec ? 2 : 1;
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_stage_forward(pulse_stage_t* s, pulse_skip_cache_t* cache, int64_t mb,
                                              const void* d_x_in, const void* d_h_in, const float* d_temb,
                                              void* d_e_out, void* d_d_out, void* stream) {
  if (!d_x_in || !d_temb || !d_d_out) return fail(PULSE_ERR_INVALID_ARG, "null x_in / temb / d_out");
  return forward_impl(s, cache, mb, d_x_in, d_h_in, const_cast<float*>(d_temb), nullptr, nullptr, d_e_out, d_d_out, stream);
}
extern "C" pulse_status_t pulse_stage_forward_temb(pulse_stage_t* s, pulse_skip_cache_t* cache, int64_t mb,
                                                   const void* d_x_in, const void* d_h_in, const int64_t* d_t,
                                                   float* d_emb, float* d_temb_stash, void* d_e_out, void* d_d_out,
                                                   void* stream) {
  if (!d_t || !d_emb || !d_temb_stash) return fail(PULSE_ERR_INVALID_ARG, "null t / emb / temb stash");
  if (!d_x_in || !d_d_out) return fail(PULSE_ERR_INVALID_ARG, "null x_in / d_out");
  return forward_impl(s, cache, mb, d_x_in, d_h_in, d_emb, d_t, d_temb_stash, d_e_out, d_d_out, stream);
}
extern "C" pulse_status_t pulse_stage_forward_enc(pulse_stage_t* s, pulse_skip_cache_t* cache, int64_t mb, const void* d_x_in,
                                                  const float* d_temb, void* d_e_out, void* stream) {
  return forward_impl(s, cache, mb, d_x_in, nullptr, const_cast<float*>(d_temb), nullptr, nullptr, d_e_out, nullptr, stream, PART_ENC);
}
extern "C" pulse_status_t pulse_stage_forward_dec(pulse_stage_t* s, pulse_skip_cache_t* cache, int64_t mb, const void* d_h_in,
                                                  void* d_d_out, void* stream) {
  return forward_impl(s, cache, mb, nullptr, d_h_in, nullptr, nullptr, nullptr, nullptr, d_d_out, stream, PART_DEC);
}

static pulse_status_t backward_impl(pulse_stage_t* s, pulse_skip_cache_t* cache, int64_t mb, const void* d_g_d_out,
                                    const void* d_g_e_out, void* d_g_x_in, void* d_g_h_in, float* d_g_temb,
                                    const float* d_temb_stash, int accumulate_wgrad, void* stream, int parts = PART_ALL,
                                    int accumulate_temb = -1) {
  pulse_status_t stt = check_bound(s, cache);
  if (stt) return stt;
  if (accumulate_temb < 0) accumulate_temb = accumulate_wgrad;
  if (parts == PART_ALL && (s->d.flags & PULSE_FLAG_SPLIT)) {      // a split stage runs its one-call backward as the two halves
    stt = backward_impl(s, cache, mb, d_g_d_out, nullptr, nullptr, d_g_h_in, d_g_temb, nullptr, accumulate_wgrad, stream, PART_DEC);
    if (stt) return stt;
    // the encoder half adds to what the decoder half (which zeroed the buffer) wrote; the timestep MLP's own gradients
    // are written by this half only and follow the caller's flag
    return backward_impl(s, cache, mb, nullptr, d_g_e_out, d_g_x_in, nullptr, d_g_temb, d_temb_stash, 1, stream, PART_ENC,
                         accumulate_wgrad);
  }
  const bool open = s->d.link == PULSE_LINK_OPEN;
  const bool enc = parts & PART_ENC, dec = parts & PART_DEC;
  if (parts != PART_ALL && !(s->d.flags & PULSE_FLAG_SPLIT)) return fail(PULSE_ERR_STATE, "the two-call forms need PULSE_FLAG_SPLIT");
  if (mb < 0 || (dec && !d_g_d_out)) return fail(PULSE_ERR_INVALID_ARG, "null g_d_out or negative mb_id");
  if (open && dec && !d_g_h_in) return fail(PULSE_ERR_INVALID_ARG, "OPEN stage needs g_h_in");
  if (!open && (d_g_h_in || d_g_e_out)) return fail(PULSE_ERR_INVALID_ARG, "CLOSED stage takes no g_h_in / g_e_out");
  int slot = -1;
  for (int i = 0; i < cache->slots; ++i) if (cache->mb[i] == mb) slot = i;
  if (slot < 0) return fail(PULSE_ERR_STATE, "backward of microbatch %lld without a live forward", (long long)mb);
  if (cache->phase[slot] != (dec ? 2 : 3))
    return fail(PULSE_ERR_STATE, "microbatch %lld: calls out of order (forward_enc, forward_dec, backward_dec, backward_enc)", (long long)mb);
  Ctx c;
  c.s = s; c.st = (cudaStream_t)stream; c.dt = s->d.dtype == PULSE_F32 ? DT_F32 : DT_BF16;
  c.skip = cache->base + (size_t)slot * cache->bytes_per_slot;
  c.work = s->d_work;
  c.stash = s->d_work + s->work_bytes + (size_t)slot * s->stash_bytes;
  c.emb = (const float*)(c.stash + s->emb_off); c.g_temb = d_g_temb; c.temb_stash = enc ? d_temb_stash : nullptr; c.acc_w = accumulate_wgrad;
  c.acc_temb = accumulate_temb; c.own_ok = dec;
  const int n_first = s->n_enc + s->n_mid, nops = (int)s->ops.size();
  c.op_lo = enc ? 0 : n_first; c.op_hi = dec ? nops : n_first;
  setup_side(s, c);
  // flipped / transposed weights for the dgrad convs, beside the memsets / column sums that open the backward (side
  // stream): first those of the last op (waited for before its dgrad), then the rest (waited for before the next op)
  int ev_wt_first = -1, ev_wt_rest = -1;
  if (!s->wt_valid) {
    c.fork();
    {
      OnSide g(c);
      prepare_weights(c, c.op_hi - 1, c.op_hi);
      if (c.side) ev_wt_first = c.mark_side();
      prepare_weights(c, 0, c.op_hi - 1);
      if (c.op_hi < nops) prepare_weights(c, c.op_hi, nops);
      if (c.side) ev_wt_rest = c.mark_side();
    }
    s->wt_valid = true;
  }
  if (dec && !accumulate_wgrad) {
    if (!s->own_valid) {
      CK_CUDA(cudaMemsetAsync((char*)s->d_grads + s->temb_grad_bytes, 0, s->grad_bytes - s->temb_grad_bytes, c.st));
    } else {                      // everything but the weight gradients that are stored whole
      for (const auto& r : s->zero_runs) CK_CUDA(cudaMemsetAsync((char*)s->d_grads + r.first, 0, r.second, c.st));
    }
  }
  CK_CUDA(cudaMemsetAsync(c.work + s->zero_begin, 0, s->zero_end - s->zero_begin, c.st));
  const bool split = parts != PART_ALL;
  const bool al = (((uintptr_t)d_g_d_out | (uintptr_t)d_g_h_in | (uintptr_t)d_g_x_in) & 255) == 0;
  if (dec) {
    if (al) { c.ov_gt[0] = s->t_dout; c.ov_gp[0] = (char*)const_cast<void*>(d_g_d_out); }       // read in place
    else CK_CUDA(cudaMemcpyAsync(c.grad(s->t_dout), d_g_d_out, c.bytes(s->t_dout), cudaMemcpyDeviceToDevice, c.st));
    if (al && open && s->t_hin != s->t_dout) { c.ov_gt[1] = s->t_hin; c.ov_gp[1] = (char*)d_g_h_in; }
  }
  // g_x_in lives in the caller's buffer only when one call writes all of it (not a per-slot skip gradient of a split stage)
  if (enc && al && d_g_x_in && s->t_xin != s->t_dout && s->t_xin != s->t_eout && !s->tensors[s->t_xin].g_in_stash) {
    c.ov_gt[2] = s->t_xin; c.ov_gp[2] = (char*)d_g_x_in;
  }
  if (enc && open) {
    if (split && s->eout_grad_by_dec) {        // the decoder half wrote the skip gradient of e_out first: g_e_out adds to it
      if (d_g_e_out) s->launches += add_inplace(c.dt, c.grad(s->t_eout), d_g_e_out, c.bytes(s->t_eout) / s->esz(), c.st);
    } else if (d_g_e_out) {
      CK_CUDA(cudaMemcpyAsync(c.grad(s->t_eout), d_g_e_out, c.bytes(s->t_eout), cudaMemcpyDeviceToDevice, c.st));
    } else {
      CK_CUDA(cudaMemsetAsync(c.grad(s->t_eout), 0, c.bytes(s->t_eout), c.st));
    }
  }
  for (int i = c.op_hi - 1; i >= c.op_lo; --i) {
    const OpPlan& op = s->ops[i];
    const int n = s->d.n;
    c.last_op = i == c.op_lo;
    if (i == c.op_hi - 1) c.wait_side(ev_wt_first);
    if (i == c.op_hi - 2) c.wait_side(ev_wt_rest);
    switch (op.kind) {
      case PULSE_OP_RESBLOCK: resblock_backward(c, op); break;
      case PULSE_OP_ATTN: attn_backward(c, op); break;
      case PULSE_OP_TBLOCK: tblock_backward(c, op); break;
      case PULSE_OP_CONV_IN:
      case PULSE_OP_DOWN: {
        const int stride = op.kind == PULSE_OP_DOWN ? 2 : 1;
        char* g_out = c.grad(op.out);
        ensure_colsum(c, op.out);
        WgradArgs w{c.dt, Cat{c.fwd(op.x0), op.cin, nullptr, 0}, n, op.hin, op.win, g_out, op.hout, op.wout, op.cout, 3,
                    stride, c.pgrad(op.p[P_C1W])};
        c.fork();
        run_wgrad(c, w);
        const bool need_gx = !(op.x0 == s->t_xin && !d_g_x_in);
        if (need_gx)
          run_dgrad(c, g_out, op.hout, op.wout, op.cout, op.wt1, 3, op.cin, c.grad(op.x0), op.acc_x0, stride, op.hin,
                    op.win);
        break;
      }
      case PULSE_OP_UP: {
        char* g_out = c.grad(op.out);
        char* g_u = c.work + s->w_gu;
        ensure_colsum(c, op.out);
        const bool wg2 = up2_wg(c, op), dg2 = up2_dg(c, op);
        c.fork();
        if (wg2) {
          run_wgrad(c, up2_wgrad_args(c, op, g_out));
        } else {          // (then the forward was the materialised form too: u exists)
          WgradArgs w{c.dt, Cat{c.fwd(op.u), op.cin, nullptr, 0}, n, op.hout, op.wout, g_out, op.hout, op.wout, op.cout, 3,
                      1, c.pgrad(op.p[P_C1W])};
          run_wgrad(c, w);
        }
        if (dg2) {
          run_conv(c, up2_dgrad_args(c, op, g_out));
        } else {
          run_dgrad(c, g_out, op.hout, op.wout, op.cout, op.wt1, 3, op.cin, g_u, 0, 1, op.hout, op.wout);
          s->launches += upsample2_bwd(c.dt, g_u, n, op.hin, op.win, op.cin, c.grad(op.x0), c.st);
        }
        break;
      }
      case PULSE_OP_HEAD: {
        char* g_out = c.grad(op.out);
        char* g_a = c.work + s->w_ga1;
        ensure_colsum(c, op.out);
        WgradArgs w{c.dt, Cat{c.fwd(op.a1), op.cin, nullptr, 0}, n, op.hin, op.win, g_out, op.hin, op.win, op.cout, 3, 1,
                    c.pgrad(op.p[P_C1W])};
        c.fork();
        run_wgrad(c, w);
        run_dgrad(c, g_out, op.hin, op.win, op.cout, op.wt1, 3, op.cin, g_a, 0, 1, op.hin, op.win);
        run_gn_bwd(c, g_a, Cat{c.fwd(op.x0), op.cin, nullptr, 0}, op.mr1, op.hin * op.win, c.par(op.p[P_GN1G]),
                   c.par(op.p[P_GN1B]), op.bst1, nullptr, c.grad(op.x0), op.cin, 0, nullptr, 0,
                   c.pgrad(op.p[P_GN1G]), c.pgrad(op.p[P_GN1B]), cs_of(c, op.x0), nullptr);
        break;
      }
    }
  }
  if (!c.tail_done) {
    if (!c.side2) c.fork();
    tail_work(c);
  }
  if (c.side2) {                               // join the tail
    cudaEvent_t e = c.new_event();
    cudaEventRecord(e, c.side2);
    cudaStreamWaitEvent(c.st, e, 0);
  }
  if (c.side) c.wait_side(c.mark_side());      // join: the caller's stream sees every weight gradient complete
  if (dec && open && c.ov_gt[1] < 0) CK_CUDA(cudaMemcpyAsync(d_g_h_in, c.grad(s->t_hin), c.bytes(s->t_hin), cudaMemcpyDeviceToDevice, c.st));
  if (enc && d_g_x_in && c.ov_gt[2] < 0) CK_CUDA(cudaMemcpyAsync(d_g_x_in, c.grad(s->t_xin), c.bytes(s->t_xin), cudaMemcpyDeviceToDevice, c.st));
  if (c.err) return fail(PULSE_ERR_CUDA, "tensor-core conv launch failed: %s", tc_last_error());
  CK_CUDA(cudaGetLastError());
  if (enc) {
    if (!s->own_valid) {          // every conv of the stage has been seen once: what is left to zero at the start of a step
      std::sort(s->own_runs.begin(), s->own_runs.end());
      s->own_runs.erase(std::unique(s->own_runs.begin(), s->own_runs.end()), s->own_runs.end());
      size_t at = s->temb_grad_bytes;
      for (const auto& r : s->own_runs) {
        if (r.first > at) s->zero_runs.push_back({at, r.first - at});
        at = r.first + r.second;
      }
      if (s->grad_bytes > at) s->zero_runs.push_back({at, s->grad_bytes - at});
      s->own_valid = true;
    }
    cache->mb[slot] = -1;
    cache->phase[slot] = 0;
    cache->live--;
  } else {
    cache->phase[slot] = 3;
  }
  s->last_was_backward = true;
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_stage_backward(pulse_stage_t* s, pulse_skip_cache_t* cache, int64_t mb,
                                               const void* d_g_d_out, const void* d_g_e_out, void* d_g_x_in,
                                               void* d_g_h_in, float* d_g_temb, int accumulate_wgrad, void* stream) {
  return backward_impl(s, cache, mb, d_g_d_out, d_g_e_out, d_g_x_in, d_g_h_in, d_g_temb, nullptr, accumulate_wgrad, stream);
}
extern "C" pulse_status_t pulse_stage_backward_temb(pulse_stage_t* s, pulse_skip_cache_t* cache, int64_t mb,
                                                    const void* d_g_d_out, const void* d_g_e_out, void* d_g_x_in,
                                                    void* d_g_h_in, float* d_g_temb, const float* d_temb_stash,
                                                    int accumulate_wgrad, void* stream) {
  if (!d_g_temb || !d_temb_stash) return fail(PULSE_ERR_INVALID_ARG, "null g_temb / temb stash");
  return backward_impl(s, cache, mb, d_g_d_out, d_g_e_out, d_g_x_in, d_g_h_in, d_g_temb, d_temb_stash, accumulate_wgrad, stream);
}
extern "C" pulse_status_t pulse_stage_backward_dec(pulse_stage_t* s, pulse_skip_cache_t* cache, int64_t mb, const void* d_g_d_out,
                                                   void* d_g_h_in, float* d_g_temb, int accumulate_wgrad, void* stream) {
  return backward_impl(s, cache, mb, d_g_d_out, nullptr, nullptr, d_g_h_in, d_g_temb, nullptr, accumulate_wgrad, stream, PART_DEC);
}
extern "C" pulse_status_t pulse_stage_backward_enc(pulse_stage_t* s, pulse_skip_cache_t* cache, int64_t mb, const void* d_g_e_out,
                                                   void* d_g_x_in, float* d_g_temb, void* stream) {
  return backward_impl(s, cache, mb, nullptr, d_g_e_out, d_g_x_in, nullptr, d_g_temb, nullptr, 1, stream, PART_ENC);
}

// ------------------------------------------------------------------------------ temb, loss
extern "C" pulse_status_t pulse_temb_stash_elems(const pulse_stage_t* s, size_t* elems) {
  if (!s || !elems) return fail(PULSE_ERR_INVALID_ARG, "null argument");
  *elems = (size_t)s->d.n * (s->d.temb_d0 + s->d.temb_dim);
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_temb_forward(pulse_stage_t* s, const int64_t* d_t, float* d_emb, float* d_stash,
                                             void* stream) {
  if (!s || !d_t || !d_emb || !d_stash) return fail(PULSE_ERR_INVALID_ARG, "null argument");
  return temb_forward_impl(s, d_t, d_emb, d_stash, (cudaStream_t)stream);
}
namespace {
pulse_status_t temb_forward_impl(pulse_stage* s, const int64_t* d_t, float* d_emb, float* d_stash, cudaStream_t st) {
  const int n = s->d.n, d0 = s->d.temb_d0, T = s->d.temb_dim;
  const int dt = s->d.dtype == PULSE_F32 ? DT_F32 : DT_BF16;
  if (s->d.temb_kind == PULSE_TEMB_SINUSOIDAL) {
    s->launches += sinusoidal(d_t, n, d0, d_emb, st);
  } else {
    if (!s->d_params) return fail(PULSE_ERR_STATE, "parameters not bound");
    float* emb0 = d_stash;
    float* z1 = d_stash + (size_t)n * d0;
    s->launches += sinusoidal(d_t, n, d0, emb0, st);
    s->launches += linear_fwd(dt, emb0, n, d0, T, s->d_params + s->params[0].off, s->d_params + s->params[1].off, 0, z1, st);
    s->launches += linear_fwd(dt, z1, n, T, T, s->d_params + s->params[2].off, s->d_params + s->params[3].off, 1, d_emb, st);
  }
  CK_CUDA(cudaGetLastError());
  return PULSE_OK;
}
}  // namespace
extern "C" pulse_status_t pulse_temb_backward(pulse_stage_t* s, const float* d_g_emb, const float* d_stash,
                                              int accumulate_wgrad, void* stream) {
  if (!s || !d_g_emb || !d_stash) return fail(PULSE_ERR_INVALID_ARG, "null argument");
  return temb_backward_impl(s, d_g_emb, d_stash, accumulate_wgrad, (cudaStream_t)stream);
}
namespace {
pulse_status_t temb_backward_impl(pulse_stage* s, const float* d_g_emb, const float* d_stash, int accumulate_wgrad,
                                  cudaStream_t st) {
  if (s->d.temb_kind == PULSE_TEMB_SINUSOIDAL) return PULSE_OK;
  if (!s->d_params || !s->d_grads || !s->d_work) return fail(PULSE_ERR_STATE, "parameters / workspace not bound");
  const int n = s->d.n, d0 = s->d.temb_d0, T = s->d.temb_dim;
  const int dt = s->d.dtype == PULSE_F32 ? DT_F32 : DT_BF16;
  if (!accumulate_wgrad) CK_CUDA(cudaMemsetAsync(s->d_grads, 0, s->temb_grad_bytes, st));
  const float* emb0 = d_stash;
  const float* z1 = d_stash + (size_t)n * d0;
  float* g_z1 = (float*)(s->d_work + s->w_tmpf);     // [n,T] fp32
  auto G = [&](int p) { return (float*)((char*)s->d_grads + s->params[p].goff); };
  // emb = W2 silu(z1) + b2
  s->launches += linear_bwd(dt, z1, d_g_emb, n, T, T, s->d_params + s->params[2].off, 1, G(2), G(3), g_z1, 0, st);
  // z1 = W1 emb0 + b1
  s->launches += linear_bwd(dt, emb0, g_z1, n, d0, T, s->d_params + s->params[0].off, 0, G(0), G(1), nullptr, 0, st);
  CK_CUDA(cudaGetLastError());
  return PULSE_OK;
}
}  // namespace
extern "C" pulse_status_t pulse_mse_fwd_bwd(int dtype, const void* d_d, const void* d_target, size_t numel, float scale,
                                            float* d_loss, void* d_g_d, void* stream) {
  if (!d_d || !d_target || !d_loss || !d_g_d) return fail(PULSE_ERR_INVALID_ARG, "null argument");
  if (dtype != PULSE_F32 && dtype != PULSE_BF16) return fail(PULSE_ERR_INVALID_ARG, "dtype");
  const int V = dtype == PULSE_F32 ? 4 : 8;
  if (numel == 0 || numel % V) return fail(PULSE_ERR_SHAPE, "numel must be a positive multiple of %d", V);
  mse_fwd_bwd(dtype == PULSE_F32 ? DT_F32 : DT_BF16, d_d, d_target, numel, scale, d_loss, d_g_d, (cudaStream_t)stream);
  CK_CUDA(cudaGetLastError());
  return PULSE_OK;
}

// ------------------------------------------------------------------------------ profiling
extern "C" pulse_status_t pulse_stage_profile(pulse_stage_t* s, int enable) {
  if (!s) return fail(PULSE_ERR_INVALID_ARG, "null stage");
  s->profiling = enable != 0;
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_stage_profile_read(pulse_stage_t* s, double ms[6], uint64_t launches[6], double flops[6],
                                                   double bytes[6]) {
  if (!s || !ms || !launches || !flops || !bytes) return fail(PULSE_ERR_INVALID_ARG, "null argument");
  for (int i = 0; i < PULSE_KCLASS_COUNT; ++i) { ms[i] = 0; launches[i] = 0; flops[i] = 0; bytes[i] = 0; }
  for (auto& sp : s->spans) {
    CK_CUDA(cudaEventSynchronize(sp.e1));
    float t = 0.f;
    CK_CUDA(cudaEventElapsedTime(&t, sp.e0, sp.e1));
    ms[sp.klass] += t; launches[sp.klass] += sp.launches; flops[sp.klass] += sp.flops; bytes[sp.klass] += sp.bytes;
    s->event_pool.push_back(sp.e0); s->event_pool.push_back(sp.e1);
  }
  s->spans.clear();
  return PULSE_OK;
}

// ------------------------------------------------------------------------------ single operators
static pulse_status_t check_conv(int dtype, int c0, int c1, int n, int h, int w, int ksize, int stride, int cout) {
  if (dtype != PULSE_F32 && dtype != PULSE_BF16) return fail(PULSE_ERR_INVALID_ARG, "dtype");
  if (n <= 0 || h <= 0 || w <= 0 || c0 <= 0 || c1 < 0 || cout <= 0) return fail(PULSE_ERR_INVALID_ARG, "non-positive size");
  if (ksize != 1 && ksize != 3) return fail(PULSE_ERR_UNSUPPORTED, "ksize must be 1 or 3");
  if (stride != 1 && stride != 2) return fail(PULSE_ERR_UNSUPPORTED, "stride must be 1 or 2");
  if (stride == 2 && ((h | w) & 1)) return fail(PULSE_ERR_SHAPE, "stride 2 needs even H, W");
  return PULSE_OK;
}
static int conv_kernel_of(int kernel) { return kernel == PULSE_CONV_TC_PAIR ? CONV_K_PAIR : kernel == PULSE_CONV_TC_1CTA ? CONV_K_1CTA : CONV_K_AUTO; }
static pulse_status_t check_kernel(int kernel, const ConvArgs& a) {
  if (kernel < PULSE_CONV_AUTO || kernel > PULSE_CONV_TC_1CTA) return fail(PULSE_ERR_INVALID_ARG, "kernel selector %d", kernel);
  if ((kernel == PULSE_CONV_TC_PAIR || kernel == PULSE_CONV_TC_1CTA) && !conv_tc_any_supported(a))
    return fail(PULSE_ERR_UNSUPPORTED, "the requested tcgen05 kernel does not cover this shape / dtype");
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_conv2d(int dtype, int kernel, const void* d_src0, int c0, const void* d_src1, int c1,
                                       int n, int h, int w, int ksize, int stride, const void* d_w, int cout,
                                       const void* d_bias, const float* d_pn, const void* d_residual, void* d_out,
                                       float* d_chan_stats, void* stream) {
  pulse_status_t s = check_conv(dtype, c0, c1, n, h, w, ksize, stride, cout);
  if (s) return s;
  if (!d_src0 || !d_w || !d_out || (c1 && !d_src1)) return fail(PULSE_ERR_INVALID_ARG, "null pointer");
  ConvArgs a;
  a.dt = dtype == PULSE_F32 ? DT_F32 : DT_BF16; a.src = Cat{d_src0, c0, d_src1, c1}; a.n = n; a.hin = h; a.win = w;
  a.hout = h / stride; a.wout = w / stride; a.ksize = ksize; a.stride = stride; a.mode = CONV_FPROP; a.w = d_w;
  a.cout = cout; a.bias = d_bias; a.pn = d_pn; a.residual = d_residual; a.out = d_out; a.accumulate = 0;
  a.kernel = conv_kernel_of(kernel);
  if ((s = check_kernel(kernel, a))) return s;
  const bool tc = kernel != PULSE_CONV_SIMT && conv_tc_any_supported(a);
  const bool fused = d_chan_stats && tc && (a.cst = d_chan_stats, conv_emits_stats(a));
  if (!fused) a.cst = nullptr;
  const int r = tc ? conv_tc_any(a, (cudaStream_t)stream) : conv_simt(a, (cudaStream_t)stream);
  if (r < 0) return fail(PULSE_ERR_CUDA, "tensor-core conv launch failed: %s", tc_last_error());
  if (d_chan_stats && !fused) chan_stats(a.dt, d_out, n, a.hout * a.wout, cout, d_chan_stats, (cudaStream_t)stream);
  CK_CUDA(cudaGetLastError());
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_conv2d_dgrad(int dtype, int kernel, const void* d_g, int n, int h, int w, int cin,
                                             int ksize, int stride, const void* d_w, int cout, void* d_wt, void* d_g_in,
                                             int accumulate, void* stream) {
  pulse_status_t s = check_conv(dtype, cin, 0, n, h, w, ksize, stride, cout);
  if (s) return s;
  if (!d_g || !d_w || !d_wt || !d_g_in) return fail(PULSE_ERR_INVALID_ARG, "null pointer");
  const int dt = dtype == PULSE_F32 ? DT_F32 : DT_BF16;
  cudaStream_t st = (cudaStream_t)stream;
  flip_transpose(dt, d_w, cout, ksize, cin, d_wt, st);
  ConvArgs a;
  a.dt = dt; a.src = Cat{d_g, cout, nullptr, 0}; a.n = n; a.hin = h / stride; a.win = w / stride; a.hout = h; a.wout = w;
  a.ksize = ksize; a.stride = 1; a.mode = stride == 2 ? CONV_DGRAD_S2 : CONV_FPROP; a.w = d_wt; a.cout = cin;
  a.bias = nullptr; a.pn = nullptr; a.residual = nullptr; a.out = d_g_in; a.accumulate = accumulate;
  a.kernel = conv_kernel_of(kernel);
  if ((s = check_kernel(kernel, a))) return s;
  const int r = (kernel != PULSE_CONV_SIMT && conv_tc_any_supported(a)) ? conv_tc_any(a, st) : conv_simt(a, st);
  if (r < 0) return fail(PULSE_ERR_CUDA, "tensor-core conv launch failed: %s", tc_last_error());
  CK_CUDA(cudaGetLastError());
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_conv2d_wgrad(int dtype, int force_simt, const void* d_src0, int c0, const void* d_src1,
                                             int c1, int n, int h, int w, int ksize, int stride, const void* d_g, int cout,
                                             float* d_dw, int accumulate, void* stream) {
  pulse_status_t s = check_conv(dtype, c0, c1, n, h, w, ksize, stride, cout);
  if (s) return s;
  if (!d_src0 || !d_g || !d_dw || (c1 && !d_src1)) return fail(PULSE_ERR_INVALID_ARG, "null pointer");
  WgradArgs a{dtype == PULSE_F32 ? DT_F32 : DT_BF16, Cat{d_src0, c0, d_src1, c1}, n, h, w, d_g, h / stride, w / stride,
              cout, ksize, stride, d_dw};
  const bool tc = !force_simt && wgrad_tc_any_supported(a);
  if (!accumulate) {
    if (tc && wgrad_whole_tiles(a)) a.overwrite = 1;
    else CK_CUDA(cudaMemsetAsync(d_dw, 0, (size_t)cout * ksize * ksize * (c0 + c1) * sizeof(float), (cudaStream_t)stream));
  }
  const int r = tc ? wgrad_tc_any(a, (cudaStream_t)stream) : wgrad_simt(a, (cudaStream_t)stream);
  if (r < 0) return fail(PULSE_ERR_CUDA, "tensor-core wgrad launch failed: %s", tc_last_error());
  CK_CUDA(cudaGetLastError());
  return PULSE_OK;
}

// ---- attention core in isolation
static pulse_status_t check_attn(int dtype, int n, int t, int c, int heads) {
  if (dtype != PULSE_F32 && dtype != PULSE_BF16) return fail(PULSE_ERR_INVALID_ARG, "dtype");
  if (n <= 0 || t <= 0 || c <= 0 || heads <= 0) return fail(PULSE_ERR_INVALID_ARG, "non-positive size");
  if (!attn_supported(c, heads)) return fail(PULSE_ERR_SHAPE, "channels %d not divisible by heads %d, or more than 128 per head", c, heads);
  return PULSE_OK;
}
extern "C" size_t pulse_attention_stats_floats(int n, int heads, int tokens) {
  return (n <= 0 || heads <= 0 || tokens <= 0) ? 0 : attn_stats_floats(n, heads, tokens);
}
extern "C" pulse_status_t pulse_attention(int dtype, int force_simt, const void* d_qkv, int n, int tokens, int c, int heads,
                                          void* d_o, float* d_stats, void* stream) {
  pulse_status_t s = check_attn(dtype, n, tokens, c, heads);
  if (s) return s;
  if (!d_qkv || !d_o || !d_stats) return fail(PULSE_ERR_INVALID_ARG, "null pointer");
  if (attn_fwd(dtype == PULSE_F32 ? DT_F32 : DT_BF16, d_qkv, n, tokens, c, heads, d_o, d_stats, (cudaStream_t)stream, !force_simt) < 0)
    return fail(PULSE_ERR_CUDA, "tensor-core attention launch failed: %s", tc_last_error());
  CK_CUDA(cudaGetLastError());
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_attention_backward(int dtype, int force_simt, const void* d_qkv, const void* d_g_o, int n,
                                                   int tokens, int c, int heads, float* d_stats, void* d_g_qkv,
                                                   void* stream) {
  pulse_status_t s = check_attn(dtype, n, tokens, c, heads);
  if (s) return s;
  if (!d_qkv || !d_g_o || !d_stats || !d_g_qkv) return fail(PULSE_ERR_INVALID_ARG, "null pointer");
  if (attn_bwd(dtype == PULSE_F32 ? DT_F32 : DT_BF16, d_qkv, d_g_o, n, tokens, c, heads, d_stats, d_g_qkv, (cudaStream_t)stream,
               !force_simt) < 0)
    return fail(PULSE_ERR_CUDA, "tensor-core attention launch failed: %s", tc_last_error());
  CK_CUDA(cudaGetLastError());
  return PULSE_OK;
}

// ---- nearest-2x upsample + 3x3 conv (row a6) as the 4-phase form, in isolation
static pulse_status_t check_up(int dtype, int kernel, int n, int h, int w, int cin, int cout) {
  if (dtype != PULSE_BF16) return fail(PULSE_ERR_UNSUPPORTED, "the 4-phase upsample conv is a tcgen05 (bf16) path");
  if (n <= 0 || h <= 0 || w <= 0 || cin <= 0 || cout <= 0) return fail(PULSE_ERR_INVALID_ARG, "non-positive size");
  if (kernel != PULSE_CONV_AUTO && kernel != PULSE_CONV_TC_PAIR && kernel != PULSE_CONV_TC_1CTA)
    return fail(PULSE_ERR_INVALID_ARG, "kernel selector %d", kernel);
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_upsample_conv2d(int dtype, int kernel, const void* d_src, int n, int h, int w, int cin,
                                                const void* d_w, int cout, const void* d_bias, void* d_wp_scratch,
                                                void* d_out, float* d_chan_stats, void* stream) {
  pulse_status_t s = check_up(dtype, kernel, n, h, w, cin, cout);
  if (s) return s;
  if (!d_src || !d_w || !d_wp_scratch || !d_out) return fail(PULSE_ERR_INVALID_ARG, "null pointer");
  cudaStream_t st = (cudaStream_t)stream;
  ConvArgs a;
  a.dt = DT_BF16; a.src = Cat{d_src, cin, nullptr, 0}; a.n = n; a.hin = h; a.win = w; a.hout = 2 * h; a.wout = 2 * w;
  a.ksize = 3; a.stride = 1; a.mode = CONV_UP2; a.w = d_wp_scratch; a.cout = cout; a.bias = d_bias; a.pn = nullptr;
  a.residual = nullptr; a.out = d_out; a.accumulate = 0; a.kernel = conv_kernel_of(kernel);
  if (!conv_tc_any_supported(a)) return fail(PULSE_ERR_UNSUPPORTED, "shape not covered by the tcgen05 conv kernels");
  up2_weights(DT_BF16, d_w, cout, cin, d_wp_scratch, nullptr, st);
  const bool fused = d_chan_stats && (a.cst = d_chan_stats, conv_emits_stats(a));
  if (!fused) a.cst = nullptr;
  if (conv_tc_any(a, st) < 0) return fail(PULSE_ERR_CUDA, "tensor-core conv launch failed: %s", tc_last_error());
  if (d_chan_stats && !fused) chan_stats(DT_BF16, d_out, n, 4 * h * w, cout, d_chan_stats, st);
  CK_CUDA(cudaGetLastError());
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_upsample_conv2d_dgrad(int dtype, int kernel, const void* d_g, int n, int h, int w, int cin,
                                                      const void* d_w, int cout, void* d_wpt_scratch, void* d_g_in,
                                                      void* stream) {
  pulse_status_t s = check_up(dtype, kernel, n, h, w, cin, cout);
  if (s) return s;
  if (!d_g || !d_w || !d_wpt_scratch || !d_g_in) return fail(PULSE_ERR_INVALID_ARG, "null pointer");
  cudaStream_t st = (cudaStream_t)stream;
  ConvArgs a;
  a.dt = DT_BF16; a.src = Cat{d_g, cout, nullptr, 0}; a.n = n; a.hin = 2 * h; a.win = 2 * w; a.hout = h; a.wout = w;
  a.ksize = 3; a.stride = 1; a.mode = CONV_UP2_DGRAD; a.w = d_wpt_scratch; a.cout = cin; a.bias = nullptr; a.pn = nullptr;
  a.residual = nullptr; a.out = d_g_in; a.accumulate = 0; a.kernel = conv_kernel_of(kernel);
  if (!conv_tc_any_supported(a)) return fail(PULSE_ERR_UNSUPPORTED, "shape not covered by the tcgen05 conv kernels");
  up2_weights(DT_BF16, d_w, cout, cin, nullptr, d_wpt_scratch, st);
  if (conv_tc_any(a, st) < 0) return fail(PULSE_ERR_CUDA, "tensor-core conv launch failed: %s", tc_last_error());
  CK_CUDA(cudaGetLastError());
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_upsample_conv2d_wgrad(int dtype, const void* d_src, int n, int h, int w, int cin,
                                                      const void* d_g, int cout, float* d_dw, void* stream) {
  pulse_status_t s = check_up(dtype, PULSE_CONV_AUTO, n, h, w, cin, cout);
  if (s) return s;
  if (!d_src || !d_g || !d_dw) return fail(PULSE_ERR_INVALID_ARG, "null pointer");
  WgradArgs a{DT_BF16, Cat{d_src, cin, nullptr, 0}, n, h, w, d_g, 2 * h, 2 * w, cout, 3, 1, d_dw};
  a.up2 = 1;
  if (!wgrad_tc_any_supported(a)) return fail(PULSE_ERR_UNSUPPORTED, "shape not covered by the tcgen05 wgrad kernel");
  if (wgrad_tc_any(a, (cudaStream_t)stream) < 0) return fail(PULSE_ERR_CUDA, "tensor-core wgrad launch failed: %s", tc_last_error());
  CK_CUDA(cudaGetLastError());
  return PULSE_OK;
}

// d_stats layout: channel stats of x0 [n][2][c0] | channel stats of x1 [n][2][c1] | mean, r [n][2][groups]
static pulse_status_t check_gn(int dtype, int c0, int c1, int n, int h, int w, int groups) {
  if (dtype != PULSE_F32 && dtype != PULSE_BF16) return fail(PULSE_ERR_INVALID_ARG, "dtype");
  if (n <= 0 || h <= 0 || w <= 0 || c0 <= 0 || c1 < 0 || groups <= 0) return fail(PULSE_ERR_INVALID_ARG, "non-positive size");
  const int vec = dtype == PULSE_F32 ? 4 : 8;
  if ((c0 + c1) % groups) return fail(PULSE_ERR_SHAPE, "channels %d not divisible by groups %d", c0 + c1, groups);
  if (c0 % vec || c1 % vec) return fail(PULSE_ERR_SHAPE, "channel counts must be multiples of %d", vec);
  if ((c0 + c1) / vec > 1024) return fail(PULSE_ERR_UNSUPPORTED, "more than %d channels", 1024 * vec);
  return PULSE_OK;
}
extern "C" size_t pulse_groupnorm_stats_floats(int n, int c, int groups) {
  if (n <= 0 || c <= 0 || groups <= 0) return 0;
  return (size_t)n * 2 * ((size_t)c + (size_t)groups);
}
extern "C" pulse_status_t pulse_groupnorm_silu(int dtype, const void* d_x0, int c0, const void* d_x1, int c1, int n, int h,
                                               int w, int groups, float eps, const void* d_gamma, const void* d_beta,
                                               float* d_stats, int reuse_stats, void* d_a, void* stream) {
  pulse_status_t s = check_gn(dtype, c0, c1, n, h, w, groups);
  if (s) return s;
  if (!d_x0 || !d_gamma || !d_beta || !d_stats || !d_a || (c1 && !d_x1)) return fail(PULSE_ERR_INVALID_ARG, "null pointer");
  const int dt = dtype == PULSE_F32 ? DT_F32 : DT_BF16, hw = h * w;
  cudaStream_t st = (cudaStream_t)stream;
  float* cst0 = d_stats;
  float* cst1 = cst0 + (size_t)n * 2 * c0;
  float* mr = cst1 + (size_t)n * 2 * c1;
  if (!reuse_stats) {
    CK_CUDA(cudaMemsetAsync(d_stats, 0, (size_t)n * 2 * (c0 + c1) * sizeof(float), st));
    chan_stats(dt, d_x0, n, hw, c0, cst0, st);
    if (c1) chan_stats(dt, d_x1, n, hw, c1, cst1, st);
  }
  gn_silu_fwd(dt, Cat{d_x0, c0, c1 ? d_x1 : nullptr, c1}, n, hw, groups, eps, d_gamma, d_beta, cst0, c1 ? cst1 : nullptr, mr,
              d_a, st);
  CK_CUDA(cudaGetLastError());
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_groupnorm_silu_backward(int dtype, int two_pass, int fwd_data_ready, const void* d_g_a,
                                                        const void* d_x0, int c0,
                                                        const void* d_x1, int c1, int n, int h, int w, int groups, float eps,
                                                        const void* d_gamma, const void* d_beta, const float* d_stats,
                                                        float* d_scratch, const void* d_add, void* d_g_x0, int accumulate0,
                                                        void* d_g_x1, int accumulate1, float* d_dgamma, float* d_dbeta,
                                                        void* stream) {
  pulse_status_t s = check_gn(dtype, c0, c1, n, h, w, groups);
  if (s) return s;
  if (!d_g_a || !d_x0 || !d_gamma || !d_beta || !d_stats || !d_scratch || !d_g_x0 || !d_dgamma || !d_dbeta ||
      (c1 && (!d_x1 || !d_g_x1)))
    return fail(PULSE_ERR_INVALID_ARG, "null pointer");
  const int dt = dtype == PULSE_F32 ? DT_F32 : DT_BF16, hw = h * w, C = c0 + c1;
  cudaStream_t st = (cudaStream_t)stream;
  const float* mr = d_stats + (size_t)n * 2 * C;
  const Cat x{d_x0, c0, c1 ? d_x1 : nullptr, c1};
  if (dt == DT_BF16 && !two_pass &&
      gn_bwd_fused(d_g_a, x, n, hw, groups, d_gamma, d_beta, mr, d_add, d_g_x0, c0, accumulate0, d_g_x1, accumulate1,
                   d_dgamma, d_dbeta, nullptr, nullptr, st, fwd_data_ready != 0) > 0) {
    CK_CUDA(cudaGetLastError());
    return PULSE_OK;
  }
  CK_CUDA(cudaMemsetAsync(d_scratch, 0, (size_t)n * 2 * C * sizeof(float), st));
  gn_silu_bwd(dt, d_g_a, x, n, hw, groups, eps, d_gamma, d_beta, mr, d_scratch, d_add, d_g_x0, c0, accumulate0, d_g_x1,
              accumulate1, d_dgamma, d_dbeta, nullptr, nullptr, st, false);
  CK_CUDA(cudaGetLastError());
  return PULSE_OK;
}
