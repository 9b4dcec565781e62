// partition.cpp - skip-aware balanced partitioning of a linearised model into p pipeline stages (host code).
// PAPER.md:L140-L197 (sec. IV-B): stage q and stage p-q+1 sit on one device; "if a skip connection exists between
// operations l_i and l_j ... and l_i is assigned to partition q, then l_j must be assigned to partition p-q+1"; minimise
// the slowest stage (Eq. 1) with the bidirectional linear-partition table of Eq. 2-5:
//   L(i', i)  = lambda (t_lat + M_a[i] / B)     + sum_{i' < l <= i} t_f[l]        encoder-side stage (i', i]
//   R(j, j')  = lambda (t_lat + M_a[j-1] / B)   + sum_{j <= l < j'} t_f[l]        decoder-side stage [j, j')
//   dp_k(i,j) = min_{i' < i, j' > j} max{ dp_{k-2}(i', j'), L(i', i), R(j, j'), c(i', i, j, j') },   target = min_i dp_p(i, i+1)
// Readings: Eq. 3/4 as printed would count operation j' twice (sum up to j' while dp(i', j') already
// covers j'..op): the decoder-side stage is [j, j').  c() = 0 iff the stage pair holds both ends of every skip it touches,
// which is a property of the two STATES: (i, j) is valid iff the skips with source <= i are exactly the skips with
// destination >= j; then c(i', i, j, j') = 0 iff (i', j') and (i, j) are valid.
// The min-max separates, min_{i'} max{L(i', i), min_{j'} max{dp(i', j'), R(j, j')}}, so a level costs O(n^3), as the
// paper's Algorithm 1 (whose text is damaged in PAPER.md) states; no monotonicity is assumed.
#include <limits>
#include <vector>

#include "../../include/pulse.h"

pulse_status_t pulse_set_error(pulse_status_t s, const char* fmt, ...);

extern "C" pulse_status_t pulse_partition(int n_ops, const double* t_f, const double* act_bytes, int n_skips,
                                          const int* skip_src, const int* skip_dst, int p, double lambda, double t_lat,
                                          double b_inter, int* cuts, double* bottleneck) {
  if (n_ops <= 0 || !t_f || p < 2 || !cuts || !bottleneck || n_skips < 0 || (n_skips && (!skip_src || !skip_dst)))
    return pulse_set_error(PULSE_ERR_INVALID_ARG, "null argument / non-positive size");
  if (p % 2) return pulse_set_error(PULSE_ERR_UNSUPPORTED, "p must be even: stages q and p-q+1 share a device");
  if (p > n_ops) return pulse_set_error(PULSE_ERR_SHAPE, "more stages (%d) than operations (%d)", p, n_ops);
  if (lambda != 0.0 && (!act_bytes || b_inter <= 0.0)) return pulse_set_error(PULSE_ERR_INVALID_ARG, "lambda != 0 needs act_bytes and b_inter > 0");
  const int n = n_ops;
  const double INF = std::numeric_limits<double>::infinity();
  for (int s = 0; s < n_skips; ++s)
    if (skip_src[s] < 1 || skip_dst[s] > n || skip_src[s] >= skip_dst[s])
      return pulse_set_error(PULSE_ERR_SHAPE, "skip %d: need 1 <= src < dst <= n_ops (1-based operation indices)", s);
  // operations are 1-based as in the paper; pre[i] = sum_{l <= i} t_f[l]
  std::vector<double> pre(n + 1, 0.0);
  for (int i = 1; i <= n; ++i) pre[i] = pre[i - 1] + t_f[i - 1];
  auto comm = [&](int l) { return lambda == 0.0 ? 0.0 : lambda * (t_lat + (l >= 1 ? act_bytes[l - 1] : 0.0) / b_inter); };
  auto Lc = [&](int i0, int i) { return comm(i) + pre[i] - pre[i0]; };                    // stage (i0, i]
  auto Rc = [&](int j, int j1) { return comm(j - 1) + pre[j1 - 1] - pre[j - 1]; };        // stage [j, j1)
  // state validity: skips with src <= i  ==  skips with dst >= j  (only "long" skips, |i - j| > 1, constrain)
  std::vector<int> csrc(n + 2, 0), cdst(n + 3, 0), mind(n + 2, n + 2);
  for (int s = 0; s < n_skips; ++s) {
    if (skip_dst[s] - skip_src[s] <= 1) continue;
    csrc[skip_src[s]]++; cdst[skip_dst[s]]++;
  }
  for (int i = 1; i <= n; ++i) csrc[i] += csrc[i - 1];
  for (int j = n; j >= 1; --j) cdst[j] += cdst[j + 1];
  {
    std::vector<int> md(n + 2, n + 2);
    for (int s = 0; s < n_skips; ++s)
      if (skip_dst[s] - skip_src[s] > 1 && skip_dst[s] < md[skip_src[s]]) md[skip_src[s]] = skip_dst[s];
    for (int i = 1; i <= n; ++i) mind[i] = md[i] < mind[i - 1] ? md[i] : mind[i - 1];
  }
  auto valid = [&](int i, int j) { return csrc[i] == cdst[j] && mind[i] >= j; };          // 0 <= i < j <= n + 1
  const int W = n + 2;
  auto at = [&](int i, int j) { return (size_t)i * W + j; };
  const int levels = p / 2;
  std::vector<std::vector<double>> dp(levels + 1, std::vector<double>((size_t)W * W, INF));
  std::vector<std::vector<int>> arg_i(levels + 1, std::vector<int>((size_t)W * W, -1)), arg_j = arg_i;
  // level 1 (k = 2 stages): the first stage (0, i] and the last stage [j, n + 1)
  for (int i = 1; i <= n; ++i)
    for (int j = i + 1; j <= n; ++j)
      if (valid(i, j)) { dp[1][at(i, j)] = Lc(0, i) > Rc(j, n + 1) ? Lc(0, i) : Rc(j, n + 1); arg_i[1][at(i, j)] = 0; arg_j[1][at(i, j)] = n + 1; }
  std::vector<double> g((size_t)W * W);
  std::vector<int> gj((size_t)W * W);
  for (int lv = 2; lv <= levels; ++lv) {
    // g(i', j) = min_{j' > j} max{dp_{lv-1}(i', j'), R(j, j')}
    for (int i0 = 1; i0 <= n; ++i0)
      for (int j = i0 + 1; j <= n; ++j) {
        double best = INF; int bj = -1;
        for (int j1 = j + 1; j1 <= n; ++j1) {
          const double a = dp[lv - 1][at(i0, j1)];
          if (a == INF) continue;
          const double r = Rc(j, j1), v = a > r ? a : r;
          if (v < best) { best = v; bj = j1; }
        }
        g[at(i0, j)] = best; gj[at(i0, j)] = bj;
      }
    for (int i = 2; i <= n; ++i)
      for (int j = i + 1; j <= n; ++j) {
        if (!valid(i, j)) continue;
        double best = INF; int bi = -1;
        for (int i0 = 1; i0 < i; ++i0) {
          const double a = g[at(i0, j)];
          if (a == INF) continue;
          const double l = Lc(i0, i), v = a > l ? a : l;
          if (v < best) { best = v; bi = i0; }
        }
        if (bi >= 0) { dp[lv][at(i, j)] = best; arg_i[lv][at(i, j)] = bi; arg_j[lv][at(i, j)] = gj[at(bi, j)]; }
      }
  }
  // target = min_i dp_p(i, i + 1)  (Eq. 5): prefix and suffix meet
  double best = INF; int bi = -1;
  for (int i = 1; i < n; ++i)
    if (dp[levels][at(i, i + 1)] < best) { best = dp[levels][at(i, i + 1)]; bi = i; }
  if (bi < 0) return pulse_set_error(PULSE_ERR_SHAPE, "no partition into %d stages satisfies the skip constraints", p);
  // back-track: cuts[m] = last operation (1-based) of stage m + 1, m = 0 .. p - 2
  int i = bi, j = bi + 1;
  for (int lv = levels; lv >= 1; --lv) {
    cuts[lv - 1] = i;                       // stage lv ends at i
    cuts[p - 1 - lv] = j - 1;               // stage p - lv ends at j - 1 (stage p - lv + 1 starts at j)
    const int ni = arg_i[lv][at(i, j)], nj = arg_j[lv][at(i, j)];
    i = ni; j = nj;
  }
  *bottleneck = best;
  return PULSE_OK;
}
