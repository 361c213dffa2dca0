// partition.cu -- memory-constrained pipeline partitioning (App. D.5).  Host code only.
//
// L sequential layers, N stages, cut points 0 = c_0 < ... < c_N = L.  Stage j (1-based) holds layers c_{j-1}+1 .. c_j and
// costs  T_j = sum t_l  and  M_j = sum s_l + w_j sum a_l  with  w_j = N - j + 1  in-flight micro-batches (Eq. 12; the
// printed "w_j = N j + 1" is garbled, P:463 fixes it: "the first stage carries N microbatches, the last carries one").
// Problem (13): minimise max_j T_j subject to M_j <= B.  Two-pass dynamic program (Eq. 15):
//   pass 1: D[i][j] = min_{j-1 <= x < i, M_j(x,i) <= B} max(D[x][j-1], T(x,i)); infeasible = +inf;
//   pass 2 (only if pass 1 is infeasible): the same recursion on pairs (overshoot, time), component-wise max,
//           lexicographic min -- "minimizes the worst overshoot first and uses the maximum stage time as a tie-breaker".
// Ties keep the FIRST minimiser x (smallest cut), so the result is deterministic.
#include <cmath>
#include <limits>
#include <vector>

#include "common.cuh"

using namespace paci;

extern "C" int paci_partition(int32_t n_layers, int32_t n_stages, const double* t, const double* s, const double* a,
                              double budget, int32_t* cuts, double* max_stage_time, double* max_overshoot) {
  const int L = n_layers, N = n_stages;
  if (!t || !s || !a || !cuts) return fail(PACI_EINVAL, "partition: null pointer");
  if (N < 1 || L < N) return fail(PACI_EINVAL, "partition: %d layers cannot fill %d stages", L, N);
  std::vector<double> pt(L + 1, 0.0), ps(L + 1, 0.0), pa(L + 1, 0.0);
  for (int l = 0; l < L; ++l) {
    if (!(t[l] >= 0.0) || !(s[l] >= 0.0) || !(a[l] >= 0.0)) return fail(PACI_EINVAL, "partition: negative or NaN profile at layer %d", l);
    pt[l + 1] = pt[l] + t[l]; ps[l + 1] = ps[l] + s[l]; pa[l + 1] = pa[l] + a[l];
  }
  const double INF = std::numeric_limits<double>::infinity();
  auto time_of = [&](int x, int i) { return pt[i] - pt[x]; };
  auto mem_of = [&](int j, int x, int i) { return (ps[i] - ps[x]) + (double)(N - j + 1) * (pa[i] - pa[x]); };
  const int W = N + 1;
  std::vector<int> arg((size_t)(L + 1) * W, -1);
  auto backtrack = [&]() {
    int i = L;
    cuts[N] = L;
    for (int j = N; j >= 1; --j) { i = arg[(size_t)i * W + j]; cuts[j - 1] = i; }
  };
  // ---- pass 1
  {
    std::vector<double> D((size_t)(L + 1) * W, INF);
    for (int i = 1; i <= L; ++i)
      if (mem_of(1, 0, i) <= budget) { D[(size_t)i * W + 1] = time_of(0, i); arg[(size_t)i * W + 1] = 0; }
    for (int j = 2; j <= N; ++j)
      for (int i = j; i <= L; ++i) {
        double best = INF; int bx = -1;
        for (int x = j - 1; x < i; ++x) {
          const double prev = D[(size_t)x * W + j - 1];
          if (prev == INF || mem_of(j, x, i) > budget) continue;
          const double v = std::fmax(prev, time_of(x, i));
          if (v < best) { best = v; bx = x; }
        }
        D[(size_t)i * W + j] = best; arg[(size_t)i * W + j] = bx;
      }
    if (D[(size_t)L * W + N] < INF) {
      backtrack();
      if (max_stage_time) *max_stage_time = D[(size_t)L * W + N];
      if (max_overshoot) *max_overshoot = 0.0;
      return 0;
    }
  }
  // ---- pass 2: (overshoot, time) pairs
  std::vector<double> Eo((size_t)(L + 1) * W, INF), Et((size_t)(L + 1) * W, INF);
  std::fill(arg.begin(), arg.end(), -1);
  auto over = [&](int j, int x, int i) { return std::fmax(0.0, mem_of(j, x, i) - budget); };
  for (int i = 1; i <= L; ++i) { Eo[(size_t)i * W + 1] = over(1, 0, i); Et[(size_t)i * W + 1] = time_of(0, i); arg[(size_t)i * W + 1] = 0; }
  for (int j = 2; j <= N; ++j)
    for (int i = j; i <= L; ++i) {
      double bo = INF, bt = INF; int bx = -1;
      for (int x = j - 1; x < i; ++x) {
        const double po = Eo[(size_t)x * W + j - 1], ptm = Et[(size_t)x * W + j - 1];
        if (po == INF && ptm == INF) continue;
        const double vo = std::fmax(po, over(j, x, i)), vt = std::fmax(ptm, time_of(x, i));
        if (vo < bo || (vo == bo && vt < bt)) { bo = vo; bt = vt; bx = x; }
      }
      Eo[(size_t)i * W + j] = bo; Et[(size_t)i * W + j] = bt; arg[(size_t)i * W + j] = bx;
    }
  backtrack();
  if (max_stage_time) *max_stage_time = Et[(size_t)L * W + N];
  if (max_overshoot) *max_overshoot = Eo[(size_t)L * W + N];
  return 1;
}
