// stage.cu - C-ABI of libpulse.so: stage descriptor -> plan -> kernel launches, and the
// skip-cache allocator.  See include/pulse.h for the contract and citations.
#include "stage.h"

#include <cstdarg>
#include <cstdio>
#include <cstring>

using namespace pulse;

// ------------------------------------------------------------------------------ errors
static thread_local char g_err[512] = "";
pulse_status_t pulse_set_error(pulse_status_t s, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof g_err, fmt, ap);
  va_end(ap);
  return s;
}

extern "C" const char* pulse_last_error(void) { return g_err; }
extern "C" int pulse_version(void) { return 100; }
extern "C" const char* pulse_status_string(pulse_status_t s) {
  switch (s) {
    case PULSE_OK: return "ok";
    case PULSE_ERR_INVALID_ARG: return "invalid argument";
    case PULSE_ERR_SHAPE: return "inconsistent shapes";
    case PULSE_ERR_UNSUPPORTED: return "unsupported";
    case PULSE_ERR_BUFFER_TOO_SMALL: return "buffer too small";
    case PULSE_ERR_CACHE: return "skip cache: slot busy, unknown microbatch or cache full";
    case PULSE_ERR_STATE: return "wrong state";
    case PULSE_ERR_CUDA: return "CUDA error";
  }
  return "unknown";
}

static size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }
static bool aligned256(const void* p) { return ((uintptr_t)p & 255) == 0; }

// ------------------------------------------------------------------------------ plan

namespace {
struct Planner {
  pulse_stage* s;
  size_t top[4] = {0, 0, 0, 0};
  size_t bump(int region, size_t bytes) {
    size_t o = top[region];
    top[region] = align256(o + bytes);
    return o;
  }
  int tensor(int region, int c, int h, int w, bool need_grad = true) {
    Tensor t;
    t.ref.region = region; t.ref.c = c; t.ref.h = h; t.ref.w = w;
    const size_t bytes = (size_t)s->d.n * h * w * c * s->esz();
    t.ref.off = bump(region, bytes);
    // split (pipeline) stages keep the gradient of a cached skip per in-flight microbatch: it is written by the backward
    // of the decoder half and read by the backward of the encoder half, with other microbatches' halves in between
    t.g_in_stash = need_grad && region == R_SKIP && (s->d.flags & PULSE_FLAG_SPLIT);
    t.goff = need_grad ? bump(t.g_in_stash ? R_STASH : R_WORK, bytes) : 0;
    s->tensors.push_back(t);
    return (int)s->tensors.size() - 1;
  }
  int param(const std::string& name, int rank, int s0, int s1 = 1, int s2 = 1, int s3 = 1) {
    ParamInfo p;
    p.name = name; p.rank = rank;
    p.shape[0] = s0; p.shape[1] = s1; p.shape[2] = s2; p.shape[3] = s3;
    p.numel = (size_t)s0 * s1 * s2 * s3;
    p.off = s->param_bytes; p.goff = s->grad_bytes;
    s->param_bytes = align256(p.off + p.numel * s->esz());
    s->grad_bytes = align256(p.goff + p.numel * 4);
    s->pindex[name] = (int)s->params.size();
    s->params.push_back(p);
    return (int)s->params.size() - 1;
  }
};
}  // namespace

static pulse_status_t build_plan(pulse_stage* s) {
  const pulse_stage_desc& d = s->d;
  Planner pl; pl.s = s;
  const int G = d.groups, T = d.temb_dim, vec = d.dtype == PULSE_F32 ? 4 : 8;
  auto chk_c = [&](int c, const char* what) -> bool { return c > 0 && c % G == 0 && c % vec == 0 && c / vec <= 512; };
  if (d.temb_kind == PULSE_TEMB_MLP) {
    pl.param("temb.w1", 2, T, d.temb_d0); pl.param("temb.b1", 1, T);
    pl.param("temb.w2", 2, T, T); pl.param("temb.b2", 1, T);
  } else if (d.temb_d0 != T) {
    return fail(PULSE_ERR_SHAPE, "sinusoidal temb needs temb_d0 == temb_dim");
  }
  s->temb_grad_bytes = s->grad_bytes;
  if (d.temb_d0 % 2) return fail(PULSE_ERR_SHAPE, "temb_d0 must be even");
  if (G > 64) return fail(PULSE_ERR_UNSUPPORTED, "at most 64 GroupNorm groups");

  std::vector<int> stack;
  int cur = pl.tensor(d.x_in_is_skip ? R_SKIP : R_STASH, d.c_in, d.h, d.w);
  s->t_xin = cur;
  if (d.x_in_is_skip) { s->skip_tensor.push_back(cur); stack.push_back(cur); }
  s->emb_off = pl.bump(R_STASH, (size_t)d.n * T * 4);

  size_t m_out = 0, m_cat = 0, m_gu = 0, m_qkv = 0, m_t4 = 0, m_tc = 0;
  auto upd = [](size_t& m, size_t v) { if (v > m) m = v; };

  auto plan_ops = [&](const std::vector<pulse_op_desc>& list, const char* phase, bool is_dec) -> pulse_status_t {
    for (size_t i = 0; i < list.size(); ++i) {
      const pulse_op_desc& o = list[i];
      OpPlan op;
      for (int k = 0; k < 16; ++k) op.p[k] = -1;
      const Tensor& tin = s->tensors[cur];
      op.kind = o.kind; op.cin = o.cin; op.cskip = o.skip_channels; op.cout = o.cout; op.heads = o.heads;
      op.hin = tin.ref.h; op.win = tin.ref.w; op.hout = op.hin; op.wout = op.win;
      op.x0 = cur;
      if (tin.ref.c != o.cin) return fail(PULSE_ERR_SHAPE, "%s%zu: cin %d but input has %d channels", phase, i, o.cin, tin.ref.c);
      const std::string pre = std::string(phase) + std::to_string(i) + ".";
      const int ctot = o.cin + o.skip_channels;
      const size_t pix = (size_t)d.n * op.hin * op.win;
      if (o.kind == PULSE_OP_RESBLOCK) {
        if (o.skip_channels > 0) {
          if (!is_dec) return fail(PULSE_ERR_SHAPE, "%s%zu: only decoder ResBlocks pop skips", phase, i);
          if (stack.empty()) return fail(PULSE_ERR_SHAPE, "%s%zu pops a skip but none is cached", phase, i);
          op.x1 = stack.back(); stack.pop_back();
          const Tensor& ts = s->tensors[op.x1];
          if (ts.ref.c != o.skip_channels || ts.ref.h != op.hin || ts.ref.w != op.win)
            return fail(PULSE_ERR_SHAPE, "%s%zu: popped skip is [%d,%d,%d], expected [%d,%d,%d]", phase, i, ts.ref.h,
                        ts.ref.w, ts.ref.c, op.hin, op.win, o.skip_channels);
          for (size_t k = 0; k < s->skip_tensor.size(); ++k) if (s->skip_tensor[k] == op.x1) op.pop = (int)k;
        }
        if (!chk_c(ctot, "cin") || !chk_c(o.cout, "cout") || o.cin % vec)
          return fail(PULSE_ERR_SHAPE, "%s%zu: channels %d|%d -> %d not divisible by groups %d / vector %d", phase, i,
                      o.cin, o.skip_channels, o.cout, G, vec);
        op.p[P_GN1G] = pl.param(pre + "gn1.gamma", 1, ctot); op.p[P_GN1B] = pl.param(pre + "gn1.beta", 1, ctot);
        op.p[P_C1W] = pl.param(pre + "conv1.w", 4, o.cout, 3, 3, ctot); op.p[P_C1B] = pl.param(pre + "conv1.b", 1, o.cout);
        op.p[P_TW] = pl.param(pre + "temb.w", 2, o.cout, T); op.p[P_TB] = pl.param(pre + "temb.b", 1, o.cout);
        op.p[P_GN2G] = pl.param(pre + "gn2.gamma", 1, o.cout); op.p[P_GN2B] = pl.param(pre + "gn2.beta", 1, o.cout);
        op.p[P_C2W] = pl.param(pre + "conv2.w", 4, o.cout, 3, 3, o.cout); op.p[P_C2B] = pl.param(pre + "conv2.b", 1, o.cout);
        if (ctot != o.cout) {
          op.p[P_SCW] = pl.param(pre + "sc.w", 4, o.cout, 1, 1, ctot); op.p[P_SCB] = pl.param(pre + "sc.b", 1, o.cout);
        }
        op.a1 = pl.tensor(R_STASH, ctot, op.hin, op.win, false);
        op.h1 = pl.tensor(R_STASH, o.cout, op.hin, op.win, false);
        op.a2 = pl.tensor(R_STASH, o.cout, op.hin, op.win, false);
        s->tensors[op.x0].gn_input = true;
        if (op.x1 >= 0) s->tensors[op.x1].gn_input = true;
        s->tensors[op.h1].gn_input = true;
        op.pn = pl.bump(R_STASH, (size_t)d.n * o.cout * 4);
        op.mr1 = pl.bump(R_STASH, (size_t)d.n * 2 * G * 4); op.mr2 = pl.bump(R_STASH, (size_t)d.n * 2 * G * 4);
        upd(m_out, pix * o.cout * s->esz()); upd(m_cat, pix * ctot * s->esz());
        op.wt1 = pl.bump(R_WORK, (size_t)o.cout * 9 * ctot * s->esz());
        op.wt2 = pl.bump(R_WORK, (size_t)o.cout * 9 * o.cout * s->esz());
        if (ctot != o.cout) op.wtsc = pl.bump(R_WORK, (size_t)o.cout * ctot * s->esz());
      } else if (o.kind == PULSE_OP_CONV_IN || o.kind == PULSE_OP_DOWN || o.kind == PULSE_OP_UP) {
        if (o.skip_channels) return fail(PULSE_ERR_SHAPE, "%s%zu: only ResBlocks pop skips", phase, i);
        if (o.kind == PULSE_OP_DOWN) {
          if (is_dec || (op.hin & 1) || (op.win & 1)) return fail(PULSE_ERR_SHAPE, "%s%zu: down needs even H,W in the encoder", phase, i);
          op.hout = op.hin / 2; op.wout = op.win / 2;
        }
        if (o.kind == PULSE_OP_UP) {
          if (!is_dec || o.cin % vec) return fail(PULSE_ERR_SHAPE, "%s%zu: up belongs to the decoder", phase, i);
          op.hout = op.hin * 2; op.wout = op.win * 2;
          op.u = pl.tensor(R_STASH, o.cin, op.hout, op.wout, false);
          upd(m_gu, (size_t)d.n * op.hout * op.wout * o.cin * s->esz());
        }
        if (o.kind == PULSE_OP_CONV_IN && is_dec) return fail(PULSE_ERR_SHAPE, "%s%zu: conv_in belongs to the encoder", phase, i);
        op.p[P_C1W] = pl.param(pre + "conv.w", 4, o.cout, 3, 3, o.cin); op.p[P_C1B] = pl.param(pre + "conv.b", 1, o.cout);
        // up: room for the 16 pre-summed (phase, tap) matrices of the 4-phase form, transposed (wt1) and plain (wt2)
        op.wt1 = pl.bump(R_WORK, (size_t)o.cout * (o.kind == PULSE_OP_UP ? 16 : 9) * o.cin * s->esz());
        if (o.kind == PULSE_OP_UP) op.wt2 = pl.bump(R_WORK, (size_t)o.cout * 16 * o.cin * s->esz());
      } else if (o.kind == PULSE_OP_ATTN) {
        // x -> GN -> xn (a1) -> 1x1 conv -> qkv (h1, 3c channels) -> attention -> o (a2) -> 1x1 conv + x -> out
        if (o.skip_channels || o.cin != o.cout || !chk_c(o.cin, "cin") || !attn_supported(o.cin, o.heads))
          return fail(PULSE_ERR_SHAPE, "%s%zu: attention needs cin == cout divisible by groups and heads, cin / heads <= 128", phase, i);
        const int c = o.cin;
        op.p[P_GN1G] = pl.param(pre + "gn.gamma", 1, c); op.p[P_GN1B] = pl.param(pre + "gn.beta", 1, c);
        op.p[P_C1W] = pl.param(pre + "qkv.w", 4, 3 * c, 1, 1, c); op.p[P_C1B] = pl.param(pre + "qkv.b", 1, 3 * c);
        op.p[P_C2W] = pl.param(pre + "proj.w", 4, c, 1, 1, c); op.p[P_C2B] = pl.param(pre + "proj.b", 1, c);
        op.a1 = pl.tensor(R_STASH, c, op.hin, op.win, false);
        op.h1 = pl.tensor(R_STASH, 3 * c, op.hin, op.win, false);
        op.a2 = pl.tensor(R_STASH, c, op.hin, op.win, false);
        s->tensors[op.x0].gn_input = true;
        op.mr1 = pl.bump(R_STASH, (size_t)d.n * 2 * G * 4);
        op.lse = pl.bump(R_STASH, attn_stats_floats(d.n, o.heads, op.hin * op.win) * 4);
        upd(m_out, pix * c * s->esz()); upd(m_cat, pix * c * s->esz()); upd(m_qkv, pix * 3 * c * s->esz());
        op.wt1 = pl.bump(R_WORK, (size_t)3 * c * c * s->esz());
        op.wt2 = pl.bump(R_WORK, (size_t)c * c * s->esz());
      } else if (o.kind == PULSE_OP_TBLOCK) {
        // [x0 | x1 -> Linear -> xs (u)] -> LN1 -> l1 (a1) -> qkv (h1) -> attention -> o (a2) -> proj + xs -> x1 (tx1)
        //   -> LN2 -> l2 (tl2) -> fc1 -> f1 (tf1) -> GELU -> g (tg) -> fc2 + x1 -> out
        const int c = o.cin;
        if (o.cin != o.cout || c % vec || !attn_supported(c, o.heads) || c > (d.dtype == PULSE_F32 ? 640 * 2 : 1280))
          return fail(PULSE_ERR_SHAPE, "%s%zu: transformer block needs cin == cout <= 1280, divisible by the vector and by heads", phase, i);
        if (o.skip_channels > 0) {
          if (!is_dec) return fail(PULSE_ERR_SHAPE, "%s%zu: only decoder-side blocks consume skips", phase, i);
          if (stack.empty()) return fail(PULSE_ERR_SHAPE, "%s%zu pops a skip but none is cached", phase, i);
          op.x1 = stack.back(); stack.pop_back();
          const Tensor& ts = s->tensors[op.x1];
          if (ts.ref.c != o.skip_channels || ts.ref.h != op.hin || ts.ref.w != op.win || o.skip_channels % vec)
            return fail(PULSE_ERR_SHAPE, "%s%zu: popped skip is [%d,%d,%d], expected [%d,%d,%d]", phase, i, ts.ref.h, ts.ref.w,
                        ts.ref.c, op.hin, op.win, o.skip_channels);
          for (size_t k = 0; k < s->skip_tensor.size(); ++k) if (s->skip_tensor[k] == op.x1) op.pop = (int)k;
          op.p[P_SCW] = pl.param(pre + "skip.w", 4, c, 1, 1, ctot); op.p[P_SCB] = pl.param(pre + "skip.b", 1, c);
          op.u = pl.tensor(R_STASH, c, op.hin, op.win, false);
          op.wtsc = pl.bump(R_WORK, (size_t)c * ctot * s->esz());
        }
        op.p[P_GN1G] = pl.param(pre + "ln1.gamma", 1, c); op.p[P_GN1B] = pl.param(pre + "ln1.beta", 1, c);
        op.p[P_C1W] = pl.param(pre + "qkv.w", 4, 3 * c, 1, 1, c); op.p[P_C1B] = pl.param(pre + "qkv.b", 1, 3 * c);
        op.p[P_C2W] = pl.param(pre + "proj.w", 4, c, 1, 1, c); op.p[P_C2B] = pl.param(pre + "proj.b", 1, c);
        op.p[P_GN2G] = pl.param(pre + "ln2.gamma", 1, c); op.p[P_GN2B] = pl.param(pre + "ln2.beta", 1, c);
        op.p[P_TW] = pl.param(pre + "fc1.w", 4, 4 * c, 1, 1, c); op.p[P_TB] = pl.param(pre + "fc1.b", 1, 4 * c);
        op.p[P_F2W] = pl.param(pre + "fc2.w", 4, c, 1, 1, 4 * c); op.p[P_F2B] = pl.param(pre + "fc2.b", 1, c);
        op.a1 = pl.tensor(R_STASH, c, op.hin, op.win, false);
        op.h1 = pl.tensor(R_STASH, 3 * c, op.hin, op.win, false);
        op.a2 = pl.tensor(R_STASH, c, op.hin, op.win, false);
        op.tx1 = pl.tensor(R_STASH, c, op.hin, op.win, false);
        op.tl2 = pl.tensor(R_STASH, c, op.hin, op.win, false);
        op.tf1 = pl.tensor(R_STASH, 4 * c, op.hin, op.win, false);
        op.tg = pl.tensor(R_STASH, 4 * c, op.hin, op.win, false);
        op.ln1 = pl.bump(R_STASH, pix * 2 * 4); op.ln2 = pl.bump(R_STASH, pix * 2 * 4);
        op.lse = pl.bump(R_STASH, attn_stats_floats(d.n, o.heads, op.hin * op.win) * 4);
        upd(m_qkv, pix * 3 * c * s->esz()); upd(m_t4, pix * 4 * c * s->esz()); upd(m_tc, pix * c * s->esz());
        upd(m_cat, pix * ctot * s->esz());
        op.wt1 = pl.bump(R_WORK, (size_t)3 * c * c * s->esz());
        op.wt2 = pl.bump(R_WORK, (size_t)c * c * s->esz());
        op.wt3 = pl.bump(R_WORK, (size_t)4 * c * c * s->esz());
        op.wt4 = pl.bump(R_WORK, (size_t)4 * c * c * s->esz());
      } else if (o.kind == PULSE_OP_HEAD) {
        if (!is_dec || o.skip_channels || !chk_c(o.cin, "cin")) return fail(PULSE_ERR_SHAPE, "%s%zu: bad head", phase, i);
        op.p[P_GN1G] = pl.param(pre + "gn.gamma", 1, o.cin); op.p[P_GN1B] = pl.param(pre + "gn.beta", 1, o.cin);
        op.p[P_C1W] = pl.param(pre + "conv.w", 4, o.cout, 3, 3, o.cin); op.p[P_C1B] = pl.param(pre + "conv.b", 1, o.cout);
        op.a1 = pl.tensor(R_STASH, o.cin, op.hin, op.win, false);
        op.mr1 = pl.bump(R_STASH, (size_t)d.n * 2 * G * 4);
        s->tensors[op.x0].gn_input = true;
        upd(m_cat, pix * o.cin * s->esz());
        op.wt1 = pl.bump(R_WORK, (size_t)o.cout * 9 * o.cin * s->esz());
      } else {
        return fail(PULSE_ERR_INVALID_ARG, "%s%zu: unknown op kind %d", phase, i, o.kind);
      }
      const bool push = !is_dec && o.push_skip;
      if (o.push_skip && (is_dec || phase[0] == 'm')) return fail(PULSE_ERR_SHAPE, "%s%zu: only encoder ops push skips", phase, i);
      op.out = pl.tensor(push ? R_SKIP : R_STASH, o.cout, op.hout, op.wout);
      s->tensors[op.out].is_out = true;
      if (push) { op.push = (int)s->skip_tensor.size(); s->skip_tensor.push_back(op.out); stack.push_back(op.out); }
      cur = op.out;
      s->ops.push_back(op);
    }
    return PULSE_OK;
  };

  pulse_status_t st = plan_ops(s->enc, "enc", false);
  if (st) return st;
  s->n_enc = (int)s->enc.size();
  if (d.link == PULSE_LINK_CLOSED) {
    for (auto& o : s->mid)
      if ((o.kind != PULSE_OP_RESBLOCK && o.kind != PULSE_OP_ATTN && o.kind != PULSE_OP_TBLOCK) || o.skip_channels)
        return fail(PULSE_ERR_SHAPE, "mid ops must be plain ResBlocks, attention or transformer blocks");
    st = plan_ops(s->mid, "mid", false);
    if (st) return st;
  } else {
    if (!s->mid.empty()) return fail(PULSE_ERR_SHAPE, "mid ops need a CLOSED stage");
    if (s->dec.empty()) return fail(PULSE_ERR_SHAPE, "OPEN stage without decoder ops");
    s->t_eout = cur;
    int hh = s->tensors[cur].ref.h, ww = s->tensors[cur].ref.w;
    if (!stack.empty()) { hh = s->tensors[stack.back()].ref.h; ww = s->tensors[stack.back()].ref.w; }
    if (s->dec[0].cin % vec) return fail(PULSE_ERR_SHAPE, "h_in channels not a multiple of %d", vec);
    cur = pl.tensor(R_STASH, s->dec[0].cin, hh, ww);
    s->t_hin = cur;
  }
  s->n_mid = (int)s->mid.size();
  st = plan_ops(s->dec, "dec", true);
  if (st) return st;
  s->n_dec = (int)s->dec.size();
  if (!stack.empty()) return fail(PULSE_ERR_SHAPE, "%zu cached skips are never popped", stack.size());
  s->t_dout = cur;

  // backward write modes: first writer of a gradient buffer stores, later writers add.  A gradient's pixel
  // sums come fused from its writers when ALL of them are GroupNorm-backward launches (norm.cu); a gradient
  // that enters from outside or is written by a conv / upsample adjoint gets a colsum pass instead.
  const bool split = (d.flags & PULSE_FLAG_SPLIT) != 0;
  if (split && d.link != PULSE_LINK_OPEN) return fail(PULSE_ERR_SHAPE, "PULSE_FLAG_SPLIT needs an OPEN stage");
  std::vector<char> written(s->tensors.size(), 0);
  written[s->t_dout] = 1; s->tensors[s->t_dout].cs_fused = false;
  // one-call form: g_e_out is written first, the skip gradient of a decoder op then adds to it.  Split form: the decoder
  // half runs BEFORE g_e_out arrives, so it is the first writer and g_e_out is added at the start of backward_enc
  if (s->t_eout >= 0) { written[s->t_eout] = split ? 0 : 1; s->tensors[s->t_eout].cs_fused = false; }
  for (int i = (int)s->ops.size() - 1; i >= 0; --i) {
    OpPlan& op = s->ops[i];
    if (split && i == s->n_enc + s->n_mid - 1 && s->t_eout >= 0) {      // the encoder half starts: g_e_out has been merged
      s->eout_grad_by_dec = written[s->t_eout] != 0;
      written[s->t_eout] = 1;
    }
    op.acc_x0 = written[op.x0]; written[op.x0] = 1;
    if (op.x1 >= 0) { op.acc_x1 = written[op.x1]; written[op.x1] = 1; }
    if (op.kind == PULSE_OP_CONV_IN || op.kind == PULSE_OP_DOWN || op.kind == PULSE_OP_UP || op.kind == PULSE_OP_TBLOCK)
      s->tensors[op.x0].cs_fused = false;
    if (op.kind == PULSE_OP_TBLOCK && op.x1 >= 0) s->tensors[op.x1].cs_fused = false;
    if ((op.kind == PULSE_OP_UP || op.kind == PULSE_OP_HEAD) && op.acc_x0)
      return fail(PULSE_ERR_UNSUPPORTED, "up/head input with a second consumer");
  }
  // split form: the pixel sums of a cached skip's gradient cannot be collected from its two writers (they run in
  // different calls): one column-sum pass over the final gradient in backward_enc instead
  if (split) for (int t : s->skip_tensor) s->tensors[t].cs_fused = false;

  // slot stash: channel stats of every tensor a GroupNorm reads, one contiguous area (zeroed per forward)
  s->cst_begin = pl.bump(R_STASH, 0);
  for (auto& t : s->tensors)
    if (t.gn_input) t.cst = pl.bump(R_STASH, (size_t)d.n * 2 * t.ref.c * 4);
  s->cst_end = pl.bump(R_STASH, 0);
  s->skip_bytes = pl.top[R_SKIP];
  s->stash_bytes = pl.top[R_STASH];
  // workspace: backward sums, one contiguous area (zeroed per backward)
  s->zero_begin = pl.bump(R_WORK, 0);
  for (auto& t : s->tensors)
    if (t.is_out) t.cs = pl.bump(R_WORK, (size_t)d.n * t.ref.c * 4);
  for (auto& op : s->ops) {
    if (op.kind == PULSE_OP_RESBLOCK) {
      op.bst1 = pl.bump(R_WORK, (size_t)d.n * 2 * (op.cin + op.cskip) * 4);
      op.bst2 = pl.bump(R_WORK, (size_t)d.n * 2 * op.cout * 4);
      op.gp = pl.bump(R_WORK, (size_t)d.n * op.cout * 4);
    } else if (op.kind == PULSE_OP_HEAD) {
      op.bst1 = pl.bump(R_WORK, (size_t)d.n * 2 * op.cin * 4);
    } else if (op.kind == PULSE_OP_ATTN) {
      op.bst1 = pl.bump(R_WORK, (size_t)d.n * 2 * op.cin * 4);
      op.gp = pl.bump(R_WORK, (size_t)d.n * 3 * op.cin * 4);       // pixel sums of g_qkv: the qkv bias gradient
    } else if (op.kind == PULSE_OP_TBLOCK) {
      // pixel sums for the bias gradients: g_xs [c] | g_qkv [3c] | g_x1 [c] | g_f1 [4c], per image
      op.gp = pl.bump(R_WORK, (size_t)d.n * 9 * op.cin * 4);
    }
  }
  s->zero_end = pl.bump(R_WORK, 0);
  s->w_ga2 = pl.bump(R_WORK, m_out); s->w_gh1 = pl.bump(R_WORK, m_out); s->w_gh1b = pl.bump(R_WORK, m_out);
  s->w_ga1 = pl.bump(R_WORK, m_cat); s->w_gsc = pl.bump(R_WORK, m_cat);
  s->w_gu = pl.bump(R_WORK, m_gu);
  s->w_gqkv = pl.bump(R_WORK, m_qkv);
  s->w_t4a = pl.bump(R_WORK, m_t4); s->w_t4b = pl.bump(R_WORK, m_t4);
  s->w_tca = pl.bump(R_WORK, m_tc); s->w_tcb = pl.bump(R_WORK, m_tc);
  s->w_tmpf = pl.bump(R_WORK, (size_t)d.n * T * 4 + 256);
  s->work_bytes = pl.top[R_WORK];
  return PULSE_OK;
}

// ------------------------------------------------------------------------------ life cycle
extern "C" pulse_status_t pulse_stage_create(const pulse_stage_desc* desc, pulse_stage_t** out) {
  if (!desc || !out) return fail(PULSE_ERR_INVALID_ARG, "null argument");
  if (desc->dtype != PULSE_F32 && desc->dtype != PULSE_BF16) return fail(PULSE_ERR_INVALID_ARG, "dtype");
  if (desc->n <= 0 || desc->h <= 0 || desc->w <= 0 || desc->c_in <= 0 || desc->groups <= 0 || desc->temb_dim <= 0 ||
      desc->max_inflight <= 0 || desc->n_enc_ops < 0 || desc->n_mid_ops < 0 || desc->n_dec_ops < 0)
    return fail(PULSE_ERR_INVALID_ARG, "non-positive size in descriptor");
  if ((desc->n_enc_ops && !desc->enc_ops) || (desc->n_mid_ops && !desc->mid_ops) || (desc->n_dec_ops && !desc->dec_ops))
    return fail(PULSE_ERR_INVALID_ARG, "null op list");
  if (desc->link != PULSE_LINK_OPEN && desc->link != PULSE_LINK_CLOSED) return fail(PULSE_ERR_INVALID_ARG, "link");
  pulse_stage* s = new (std::nothrow) pulse_stage();
  if (!s) return fail(PULSE_ERR_INVALID_ARG, "out of host memory");
  s->d = *desc;
  s->enc.assign(desc->enc_ops, desc->enc_ops + desc->n_enc_ops);
  s->mid.assign(desc->mid_ops, desc->mid_ops + desc->n_mid_ops);
  s->dec.assign(desc->dec_ops, desc->dec_ops + desc->n_dec_ops);
  s->d.enc_ops = s->enc.data(); s->d.mid_ops = s->mid.data(); s->d.dec_ops = s->dec.data();
  pulse_status_t st = build_plan(s);
  if (st) { delete s; return st; }
  *out = s;
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_stage_destroy(pulse_stage_t* s) {
  if (s) {
    for (auto& sp : s->spans) { cudaEventDestroy(sp.e0); cudaEventDestroy(sp.e1); }
    for (auto ev : s->event_pool) cudaEventDestroy(ev);
    for (auto ev : s->sync_events) cudaEventDestroy(ev);
    if (s->side) cudaStreamDestroy(s->side);
    if (s->side2) cudaStreamDestroy(s->side2);
  }
  delete s;
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_stage_param_count(const pulse_stage_t* s, int* count) {
  if (!s || !count) return fail(PULSE_ERR_INVALID_ARG, "null argument");
  *count = (int)s->params.size();
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_stage_param_info(const pulse_stage_t* s, int i, const char** name, int* rank, int shape[4],
                                                 size_t* off, size_t* goff) {
  if (!s) return fail(PULSE_ERR_INVALID_ARG, "null stage");
  if (i < 0 || i >= (int)s->params.size()) return fail(PULSE_ERR_INVALID_ARG, "param index %d out of range", i);
  const ParamInfo& p = s->params[i];
  if (name) *name = p.name.c_str();
  if (rank) *rank = p.rank;
  if (shape) for (int k = 0; k < 4; ++k) shape[k] = p.shape[k];
  if (off) *off = p.off;
  if (goff) *goff = p.goff;
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_stage_param_bytes(const pulse_stage_t* s, size_t* pb, size_t* gb) {
  if (!s) return fail(PULSE_ERR_INVALID_ARG, "null stage");
  if (pb) *pb = s->param_bytes;
  if (gb) *gb = s->grad_bytes;
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_stage_bind_params(pulse_stage_t* s, const void* d_params, float* d_grads) {
  if (!s || !d_params || !d_grads) return fail(PULSE_ERR_INVALID_ARG, "null argument");
  if (!aligned256(d_params) || !aligned256(d_grads)) return fail(PULSE_ERR_INVALID_ARG, "buffers must be 256-byte aligned");
  s->d_params = (const char*)d_params; s->d_grads = d_grads;
  s->wt_valid = false; s->wp_valid = false;
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_stage_workspace_bytes(const pulse_stage_t* s, size_t* per_stage, size_t* per_inflight) {
  if (!s) return fail(PULSE_ERR_INVALID_ARG, "null stage");
  if (per_stage) *per_stage = s->work_bytes;
  if (per_inflight) *per_inflight = s->stash_bytes;
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_stage_bind_workspace(pulse_stage_t* s, void* d, size_t bytes) {
  if (!s || !d) return fail(PULSE_ERR_INVALID_ARG, "null argument");
  if (!aligned256(d)) return fail(PULSE_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
  const size_t need = s->work_bytes + (size_t)s->d.max_inflight * s->stash_bytes;
  if (bytes < need) return fail(PULSE_ERR_BUFFER_TOO_SMALL, "workspace %zu < %zu bytes", bytes, need);
  s->d_work = (char*)d; s->work_bound = bytes;
  s->wt_valid = false; s->wp_valid = false;
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_stage_launch_count(const pulse_stage_t* s, uint64_t* n) {
  if (!s || !n) return fail(PULSE_ERR_INVALID_ARG, "null argument");
  *n = s->launches;
  return PULSE_OK;
}

// ------------------------------------------------------------------------------ skip cache
extern "C" pulse_status_t pulse_skip_cache_bytes(const pulse_stage_t* s, size_t* b) {
  if (!s || !b) return fail(PULSE_ERR_INVALID_ARG, "null argument");
  *b = s->skip_bytes;
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_skip_cache_create(pulse_stage_t* s, void* d_mem, size_t bytes, int slots,
                                                  pulse_skip_cache_t** out) {
  if (!s || !out || (!d_mem && s->skip_bytes)) return fail(PULSE_ERR_INVALID_ARG, "null argument");
  if (!aligned256(d_mem)) return fail(PULSE_ERR_INVALID_ARG, "cache memory must be 256-byte aligned");
  if (slots <= 0 || slots > s->d.max_inflight) return fail(PULSE_ERR_INVALID_ARG, "slots %d not in [1, max_inflight=%d]", slots, s->d.max_inflight);
  if (bytes < (size_t)slots * s->skip_bytes) return fail(PULSE_ERR_BUFFER_TOO_SMALL, "cache %zu < %zu bytes", bytes, (size_t)slots * s->skip_bytes);
  pulse_skip_cache* c = new (std::nothrow) pulse_skip_cache();
  if (!c) return fail(PULSE_ERR_INVALID_ARG, "out of host memory");
  c->stage = s; c->base = (char*)d_mem; c->slots = slots; c->bytes_per_slot = s->skip_bytes;
  c->mb.assign(slots, -1);
  c->phase.assign(slots, 0);
  *out = c;
  return PULSE_OK;
}
static int find_slot(const pulse_skip_cache* c, int64_t mb) {
  for (int i = 0; i < c->slots; ++i) if (c->mb[i] == mb) return i;
  return -1;
}
extern "C" pulse_status_t pulse_skip_cache_count(const pulse_skip_cache_t* c, int* n) {
  if (!c || !n) return fail(PULSE_ERR_INVALID_ARG, "null argument");
  *n = (int)c->stage->skip_tensor.size();
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_skip_cache_get(const pulse_skip_cache_t* c, int64_t mb, int k, void** d_ptr, int shape[4]) {
  if (!c || mb < 0) return fail(PULSE_ERR_INVALID_ARG, "null cache / negative microbatch id");
  const int slot = find_slot(c, mb);
  if (slot < 0) return fail(PULSE_ERR_CACHE, "microbatch %lld is not live", (long long)mb);
  if (k < 0 || k >= (int)c->stage->skip_tensor.size()) return fail(PULSE_ERR_INVALID_ARG, "skip index %d out of range", k);
  const TRef& r = c->stage->tensors[c->stage->skip_tensor[k]].ref;
  if (d_ptr) *d_ptr = c->base + (size_t)slot * c->bytes_per_slot + r.off;
  if (shape) { shape[0] = c->stage->d.n; shape[1] = r.h; shape[2] = r.w; shape[3] = r.c; }
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_skip_cache_release(pulse_skip_cache_t* c, int64_t mb) {
  if (!c || mb < 0) return fail(PULSE_ERR_INVALID_ARG, "null cache / negative microbatch id");
  const int slot = find_slot(c, mb);
  if (slot < 0) return fail(PULSE_ERR_CACHE, "microbatch %lld is not live", (long long)mb);
  c->mb[slot] = -1; c->live--;
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_skip_cache_stats(const pulse_skip_cache_t* c, int* live, size_t* live_bytes, size_t* peak) {
  if (!c) return fail(PULSE_ERR_INVALID_ARG, "null cache");
  if (live) *live = c->live;
  if (live_bytes) *live_bytes = (size_t)c->live * c->bytes_per_slot;
  if (peak) *peak = c->peak_bytes;
  return PULSE_OK;
}
extern "C" pulse_status_t pulse_skip_cache_destroy(pulse_skip_cache_t* c) {
  delete c;
  return PULSE_OK;
}
