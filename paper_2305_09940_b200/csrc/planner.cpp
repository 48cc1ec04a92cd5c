// planner.cpp — host-side cost model and plan search of osdp-b200 (no CUDA in this file).
//
// Cost model: PAPER.md:84-86 (M_i), PAPER.md:92-94 (T_i), PAPER.md:167 (size / slice_granularity);
// search: Algorithm 1 with the Search Engine's depth-first traversal and its two
// prunings.  Readings P1-P9 are listed in DESIGN.md.
//
// Times are compared as integer picoseconds (reading P9): each T_i is rounded once to an int64 count
// of 1e-12 s, so sums, ties and bounds are exact and the traversal order alone decides among equal plans.
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

#include "../../include/osdp.h"

namespace {

constexpr double kPsPerSecond = 1e12;
constexpr uint64_t kNodeBudget = 400ull * 1000 * 1000;

inline uint64_t ceil_div_u64(uint64_t a, uint64_t b) { return (a + b - 1) / b; }

struct OptionCost {
  uint64_t persist;
  uint64_t transient;
  int64_t ps;
};

// One operator cut into k slices of which z run in ZDP mode and k - z in DP mode ("partition the
// operator into 4 slices and process 1 of them in the ZDP mode and 3 of them in the DP mode"; reading P10).
// Each slice carries 1/k of the operator's parameters and model states: the ZDP slices hold ceil(model z / k)
// bytes, sharded N ways; communication is 2 collectives' worth for a DP slice and 3 for a ZDP slice
// (PAPER.md:92-94), i.e. (2 + z/k) (N-1)(alpha + S beta / N) for the operator.  z = 0 and z = k are the
// paper's pure DP and ZDP formulas exactly.
bool eval_mixed(const osdp_op_cost& op, int32_t k, int32_t z, int64_t batch, const osdp_device& dev,
                uint64_t* persist, uint64_t* transient, double* seconds) {
  if (k < 1 || z < 0 || z > k || batch < 0 || dev.N < 1) return false;
  const bool ckpt = dev.checkpointing != 0;   // PAPER.md:51, :251-253 (reading P12)
  if (ckpt && (!(dev.recompute_fraction >= 0.0) || !(dev.act_keep_fraction >= 0.0) || !(dev.act_keep_fraction <= 1.0))) return false;
  const uint64_t zdp_share = (uint64_t)(((unsigned __int128)op.model_bytes * (uint64_t)z + (uint64_t)k - 1) / (uint64_t)k);
  const uint64_t model = (op.model_bytes - zdp_share) + ceil_div_u64(zdp_share, (uint64_t)dev.N);
  uint64_t act = (uint64_t)batch * op.act_bytes;
  if (ckpt) act = (uint64_t)std::ceil((double)act * dev.act_keep_fraction);   // only the checkpoints stay resident
  if (persist) *persist = model + act + op.extra_fixed + ceil_div_u64(op.extra_summed, (uint64_t)k);
  if (transient) *transient = ceil_div_u64(op.extra_transient, (uint64_t)k);
  if (seconds) {
    // a ZDP slice: 3 collectives, 4 with checkpointing (one more gather round for the recomputation)
    const double c = 2.0 + (ckpt ? 2.0 : 1.0) * (double)z / (double)k;
    const double compute = (double)batch * op.gamma * (ckpt ? 1.0 + dev.recompute_fraction : 1.0);
    *seconds = c * (double)(dev.N - 1) * (dev.alpha + op.S * dev.beta / (double)dev.N) + compute + (double)(k - 1) * op.delta;
  }
  return true;
}

bool eval(const osdp_op_cost& op, int mode, int32_t k, int64_t batch, const osdp_device& dev,
          uint64_t* persist, uint64_t* transient, double* seconds) {
  if (mode != OSDP_DP && mode != OSDP_ZDP) return false;
  return eval_mixed(op, k, mode == OSDP_ZDP ? k : 0, batch, dev, persist, transient, seconds);
}

struct Option {
  int32_t k, z;   // k slices, z of them in ZDP mode
};
// Pure modes, in the order of reading P5: DP before ZDP, k ascending.
std::vector<Option> pure_options(const int32_t* cand, int32_t n_cand) {
  std::vector<Option> o;
  for (int m = 0; m < 2; ++m)
    for (int i = 0; i < n_cand; ++i) o.push_back({cand[i], m == 0 ? 0 : cand[i]});
  return o;
}
// Slice-level mixing, in the order of reading P10: k ascending, then z ascending (least split, DP-most first).
std::vector<Option> mixed_options(const int32_t* cand, int32_t n_cand) {
  std::vector<Option> o;
  for (int i = 0; i < n_cand; ++i)
    for (int32_t z = 0; z <= cand[i]; ++z) o.push_back({cand[i], z});
  return o;
}

inline int64_t to_ps(double seconds) { return (int64_t)std::floor(seconds * kPsPerSecond + 0.5); }

// Lagrangian lower bound on the time of the operators still to be decided, given the bytes R they may still
// use (a safe strengthening of the paper's time pruning): for any lambda >= 0,
//   sum_j t_j  >=  sum_j min_o (t_jo + lambda m_jo) - lambda R.
// lambda runs over a fixed grid num/8 * 2^e (picoseconds per byte); everything is exact in 128-bit integers
// scaled by 2^27, so a subtree is discarded only when it provably cannot beat the incumbent.
typedef __int128 i128;
constexpr int kLamExpMin = -24, kLamExpMax = 16, kLamScaleBits = 27;
constexpr int kNumLambda = (kLamExpMax - kLamExpMin + 1) * 8;
inline i128 lambda_scaled(int idx) {   // lambda * 2^27
  const int e = kLamExpMin + idx / 8, num = 8 + idx % 8;
  return (i128)num << (e - kLamExpMin);                    // num/8 * 2^e * 2^27 = num * 2^(e + 24)
}

struct Search {
  int n = 0, n_opt = 0;
  std::vector<OptionCost> cost;          // [n][n_opt]
  std::vector<uint64_t> suf_persist;     // [n+1] sum over j >= i of min_o persist
  std::vector<int64_t> suf_ps;           // [n+1]
  std::vector<i128> suf_lag;             // [n+1][kNumLambda]
  std::vector<int> prev_same;            // most recent identical operator, or -1
  std::vector<int> choice, best_choice;
  uint64_t limit = 0;
  int64_t best_ps = std::numeric_limits<int64_t>::max();
  uint64_t best_mem = 0;
  bool found = false;
  uint64_t nodes = 0;
  bool exhausted = false;

  const OptionCost& c(int i, int o) const { return cost[(size_t)i * n_opt + o]; }

  void dfs(int i, uint64_t persist, uint64_t trans, int64_t ps) {
    if (i == n) {
      // Algorithm 1 line 8: feasible and strictly faster than the incumbent.
      if (persist + trans <= limit && ps < best_ps) {
        best_ps = ps;
        best_mem = persist + trans;
        best_choice = choice;
        found = true;
      }
      return;
    }
    const int o_min = prev_same[i] >= 0 ? choice[prev_same[i]] : 0;   // canonical order among identical operators
    for (int o = o_min; o < n_opt; ++o) {
      if (++nodes > kNodeBudget) { exhausted = true; return; }
      const OptionCost& oc = c(i, o);
      const uint64_t p = persist + oc.persist;
      const uint64_t t = trans > oc.transient ? trans : oc.transient;
      // pruning 1: memory already over the limit, counting the least the rest can take
      if (p + suf_persist[i + 1] + t > limit) continue;
      const int64_t s = ps + oc.ps;
      // pruning 2: time cannot beat the best plan so far
      if (s + suf_ps[i + 1] >= best_ps) continue;
      if (i + 1 < n && best_ps != std::numeric_limits<int64_t>::max()) {
        const i128 R = (i128)(limit - p - t);              // bytes the remaining operators may still add
        const i128* L = &suf_lag[(size_t)(i + 1) * kNumLambda];
        // the dual function lambda -> L(lambda) - lambda R is concave: bisect on its slope over the grid
        auto f = [&](int l) { return L[l] - R * lambda_scaled(l); };
        int lo = 0, hi = kNumLambda - 1;
        while (lo < hi) {
          const int mid = (lo + hi) / 2;
          if (f(mid) < f(mid + 1)) lo = mid + 1; else hi = mid;
        }
        const i128 lb = f(lo) >> kLamScaleBits;                             // floor: still a lower bound
        const bool cut = lb > 0 && (i128)s + lb >= (i128)best_ps;
        if (cut) continue;
      }
      choice[i] = o;
      dfs(i + 1, p, t, s);
      if (exhausted) return;
    }
  }
};

int run_search(const osdp_op_cost* ops, int32_t n, const osdp_device* dev, int64_t batch,
               const std::vector<Option>& options, Search& S) {
  S.n = n;
  S.n_opt = (int)options.size();
  S.limit = dev->mem_limit_bytes;
  S.cost.resize((size_t)n * S.n_opt);
  for (int i = 0; i < n; ++i)
    for (int o = 0; o < S.n_opt; ++o) {
      OptionCost& oc = S.cost[(size_t)i * S.n_opt + o];
      double sec = 0;
      if (!eval_mixed(ops[i], options[o].k, options[o].z, batch, *dev, &oc.persist, &oc.transient, &sec))
        return OSDP_ERR_ARG;
      if (!(sec >= 0) || sec > 9e6) return OSDP_ERR_ARG;
      oc.ps = to_ps(sec);
    }
  S.suf_persist.assign(n + 1, 0);
  S.suf_ps.assign(n + 1, 0);
  for (int i = n - 1; i >= 0; --i) {
    uint64_t mp = std::numeric_limits<uint64_t>::max();
    int64_t mt = std::numeric_limits<int64_t>::max();
    for (int o = 0; o < S.n_opt; ++o) {
      mp = S.c(i, o).persist < mp ? S.c(i, o).persist : mp;
      mt = S.c(i, o).ps < mt ? S.c(i, o).ps : mt;
    }
    S.suf_persist[i] = S.suf_persist[i + 1] + mp;
    S.suf_ps[i] = S.suf_ps[i + 1] + mt;
  }
  S.suf_lag.assign((size_t)(n + 1) * kNumLambda, 0);
  for (int i = n - 1; i >= 0; --i)
    for (int l = 0; l < kNumLambda; ++l) {
      const i128 lam = lambda_scaled(l);
      i128 best = 0;
      for (int o = 0; o < S.n_opt; ++o) {
        const i128 v = ((i128)S.c(i, o).ps << kLamScaleBits) + (i128)S.c(i, o).persist * lam;
        if (o == 0 || v < best) best = v;
      }
      S.suf_lag[(size_t)i * kNumLambda + l] = S.suf_lag[(size_t)(i + 1) * kNumLambda + l] + best;
    }
  // Starting incumbent: the best feasible plan among the per-lambda minimisers.  It only tightens pruning 2;
  // the incumbent TIME is set one picosecond above it, so the traversal still returns the first plan (in
  // traversal order) that attains the optimum.
  {
    for (int l = -1; l < kNumLambda; ++l) {
      uint64_t persist = 0, trans = 0;
      int64_t ps = 0;
      for (int i = 0; i < n; ++i) {
        int bo = 0;
        i128 bv = 0;
        for (int o = 0; o < S.n_opt; ++o) {
          const i128 v = ((i128)S.c(i, o).ps << kLamScaleBits) + (l < 0 ? (i128)0 : (i128)S.c(i, o).persist * lambda_scaled(l)) +
                         (l < 0 ? (i128)0 : (i128)S.c(i, o).transient * lambda_scaled(l));
          if (o == 0 || v < bv) { bv = v; bo = o; }
        }
        persist += S.c(i, bo).persist;
        trans = S.c(i, bo).transient > trans ? S.c(i, bo).transient : trans;
        ps += S.c(i, bo).ps;
      }
      if (persist + trans <= S.limit && ps < S.best_ps - 1) S.best_ps = ps + 1;
    }
  }
  S.prev_same.assign(n, -1);
  for (int i = 1; i < n; ++i)
    for (int j = i - 1; j >= 0; --j)
      if (std::memcmp(&ops[i], &ops[j], sizeof(osdp_op_cost)) == 0) { S.prev_same[i] = j; break; }
  S.choice.assign(n, 0);
  S.dfs(0, 0, 0, 0);
  if (S.exhausted) return OSDP_ERR_SEARCH_LIMIT;
  return S.found ? OSDP_OK : OSDP_ERR_INFEASIBLE;
}

int check_plan_args(const osdp_op_cost* ops, int32_t n, const osdp_device* dev, const int32_t* cand,
                    int32_t n_cand, const int32_t* k_out, const int32_t* mode_out) {
  if (!ops || !dev || !cand || !k_out || !mode_out) return OSDP_ERR_NULL;
  if (n < 1 || n_cand < 1 || n_cand > 64 || dev->N < 1) return OSDP_ERR_ARG;
  for (int i = 0; i < n_cand; ++i)
    if (cand[i] < 1 || (i > 0 && cand[i] <= cand[i - 1])) return OSDP_ERR_ARG;
  return OSDP_OK;
}

}  // namespace

extern "C" {

int osdp_cost_eval(const osdp_op_cost* op, int mode, int32_t k, int64_t batch, const osdp_device* dev,
                   uint64_t* persist_bytes, uint64_t* transient_bytes, double* seconds) {
  if (!op || !dev) return OSDP_ERR_NULL;
  return eval(*op, mode, k, batch, *dev, persist_bytes, transient_bytes, seconds) ? OSDP_OK : OSDP_ERR_ARG;
}

int osdp_plan(const osdp_op_cost* ops, int32_t n, const osdp_device* dev, int64_t batch,
              const int32_t* k_candidates, int32_t n_cand,
              int32_t* k_out, int32_t* mode_out, double* est_seconds, uint64_t* est_peak_bytes) {
  int st = check_plan_args(ops, n, dev, k_candidates, n_cand, k_out, mode_out);
  if (st != OSDP_OK) return st;
  if (batch < 0) return OSDP_ERR_ARG;
  Search S;
  const std::vector<Option> options = pure_options(k_candidates, n_cand);
  st = run_search(ops, n, dev, batch, options, S);
  if (st != OSDP_OK) return st;
  for (int i = 0; i < n; ++i) {
    mode_out[i] = options[S.best_choice[i]].z == 0 ? OSDP_DP : OSDP_ZDP;
    k_out[i] = options[S.best_choice[i]].k;
  }
  if (est_seconds) *est_seconds = (double)S.best_ps / kPsPerSecond;
  if (est_peak_bytes) *est_peak_bytes = S.best_mem;
  return OSDP_OK;
}

int osdp_cost_eval_mixed(const osdp_op_cost* op, int32_t k, int32_t zdp_slices, int64_t batch, const osdp_device* dev,
                         uint64_t* persist_bytes, uint64_t* transient_bytes, double* seconds) {
  if (!op || !dev) return OSDP_ERR_NULL;
  return eval_mixed(*op, k, zdp_slices, batch, *dev, persist_bytes, transient_bytes, seconds) ? OSDP_OK : OSDP_ERR_ARG;
}

int osdp_plan_mixed(const osdp_op_cost* ops, int32_t n, const osdp_device* dev, int64_t batch,
                    const int32_t* k_candidates, int32_t n_cand,
                    int32_t* k_out, int32_t* zdp_slices_out, double* est_seconds, uint64_t* est_peak_bytes) {
  int st = check_plan_args(ops, n, dev, k_candidates, n_cand, k_out, zdp_slices_out);
  if (st != OSDP_OK) return st;
  if (batch < 0) return OSDP_ERR_ARG;
  for (int i = 0; i < n_cand; ++i)
    if (k_candidates[i] > 1024) return OSDP_ERR_ARG;   // the option table has k + 1 entries per candidate
  Search S;
  const std::vector<Option> options = mixed_options(k_candidates, n_cand);
  st = run_search(ops, n, dev, batch, options, S);
  if (st != OSDP_OK) return st;
  for (int i = 0; i < n; ++i) {
    k_out[i] = options[S.best_choice[i]].k;
    zdp_slices_out[i] = options[S.best_choice[i]].z;
  }
  if (est_seconds) *est_seconds = (double)S.best_ps / kPsPerSecond;
  if (est_peak_bytes) *est_peak_bytes = S.best_mem;
  return OSDP_OK;
}

int osdp_plan_batch(const osdp_op_cost* ops, int32_t n, const osdp_device* dev, int64_t batch_max,
                    const int32_t* k_candidates, int32_t n_cand,
                    int32_t* k_out, int32_t* mode_out, int64_t* batch_out,
                    double* est_seconds, uint64_t* est_peak_bytes) {
  int st = check_plan_args(ops, n, dev, k_candidates, n_cand, k_out, mode_out);
  if (st != OSDP_OK) return st;
  if (!batch_out) return OSDP_ERR_NULL;
  if (batch_max < 1) return OSDP_ERR_ARG;
  // Algorithm 1: candidates (T*(b), p*(b), b) for b = 1, 2, 3, ...; break at the first infeasible b;
  // final argmin of the per-sample time T(b)/b (Eq. 1), first b wins ties.
  bool any = false;
  int64_t best_b = 0, best_ps = 0;
  uint64_t best_mem = 0;
  std::vector<int> best_choice;
  const std::vector<Option> options = pure_options(k_candidates, n_cand);
  for (int64_t b = 1; b <= batch_max; ++b) {
    Search S;
    st = run_search(ops, n, dev, b, options, S);
    if (st == OSDP_ERR_INFEASIBLE) break;
    if (st != OSDP_OK) return st;
    // compare S.best_ps / b  <  best_ps / best_b  exactly: cross-multiply in 128-bit
    const bool better = !any || ((__int128)S.best_ps * best_b < (__int128)best_ps * b);
    if (better) {
      any = true;
      best_b = b; best_ps = S.best_ps; best_mem = S.best_mem; best_choice = S.best_choice;
    }
  }
  if (!any) return OSDP_ERR_INFEASIBLE;
  for (int i = 0; i < n; ++i) {
    mode_out[i] = options[best_choice[i]].z == 0 ? OSDP_DP : OSDP_ZDP;
    k_out[i] = options[best_choice[i]].k;
  }
  *batch_out = best_b;
  if (est_seconds) *est_seconds = (double)best_ps / kPsPerSecond;
  if (est_peak_bytes) *est_peak_bytes = best_mem;
  return OSDP_OK;
}

}  // extern "C"
