// fg_batch.cpp — several graphs integrated "simultaneously" (Sec. IV.C):
//   initialisation stage  a fixed number of samples per graph gives first values of sigma_down,j and of t_j, the time per sample;
//   acceptance (18)       abs_tol_j = (1/4) sigma_down,j sqrt(sum_l sigma_down,l^2) / sum_l sigma_down,l, floating with N;
//   block scheduling      the graph of the next block is drawn with p_j = (C_j / sqrt t_j) / sum_l (C_l / sqrt t_l),
//                         C_j = sigma_j sqrt N_j  (the paper uses its sigma_up here, an error estimate defined only in its
//                         Ref. [32]; sigma_down of (17) stands in, and the paper's "little modification for stabilization" is
//                         not described and not applied);
//   combination (19)      sigma^2 = sum_j sigma_j^2, value = sum_j mean_j.
// Host logic only, written on top of the C ABI of fg.h (the kernels are reached through fg_integrate_range).  The draw of a
// block's graph uses Philox4x32-10 with key = scheduler seed and counter = block index, so a schedule is reproducible from
// (seed, the folded results, the times t_j); next/fold are separate calls so that several ranks can run one schedule:
// every rank draws the same blocks, integrates its own, and folds all of them in block order (paper_1909_08015_b200/dist.py).
#include <cmath>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/fg.h"

namespace {

void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1, uint32_t out[4]) {
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    c1 = (uint32_t)p1; c3 = (uint32_t)p0; c0 = n0; c2 = n2;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
double uniform53(uint32_t w0, uint32_t w1) { return ((double)((((uint64_t)w0 << 32) | w1) >> 11) + 0.5) * 0x1p-53; }

struct GraphState {
  fg_plan* plan = nullptr;
  fg_result sum;              // running sums of everything folded so far (pilot included)
  bool has = false;
  uint64_t next_sample = 0;   // first Philox sample id not yet handed out
  double t = 1.0;             // seconds per sample
  double abs_tol = 0.0;
  int32_t kmm[3] = {-1, -1, -1};   // gauge-invariant class, set by fg_batch_set_classes
};

}  // namespace

struct fg_batch {
  std::vector<GraphState> g;
  double rel_tol = 0.0, target = 0.0;
  uint64_t blocks_drawn = 0;
};

int fg_internal_fail(int code, const std::string& m);      // fg_kernels.cu: sets fg_last_error_message()
static int bfail(int code, const std::string& m) { return fg_internal_fail(code, m); }

// per-sample standard deviation s_j = sigma_down,j sqrt(N_j), from (17)
static double per_sample_sigma(const fg_result& r) {
  if (r.n_samples == 0) return 0.0;
  const double v = r.variance * (double)r.n_samples;
  return v > 0.0 ? std::sqrt(v) : 0.0;
}

// (18): sigma_down,l = s_l / sqrt(N_l), with N_l = target samples per graph if a target is set (a projection to the end of
// the run), else the samples folded so far
static void update_tolerances(fg_batch* b) {
  const size_t n = b->g.size();
  std::vector<double> sig(n, 0.0); double s1 = 0.0, s2 = 0.0;
  for (size_t j = 0; j < n; ++j) {
    const fg_result& r = b->g[j].sum;
    const double N = b->target > 0.0 ? b->target : (double)r.n_samples;
    sig[j] = N > 0.0 ? per_sample_sigma(r) / std::sqrt(N) : 0.0;
    s1 += sig[j]; s2 += sig[j] * sig[j];
  }
  for (size_t j = 0; j < n; ++j) b->g[j].abs_tol = s1 > 0.0 ? 0.25 * sig[j] * std::sqrt(s2) / s1 : 0.0;
}

static void probabilities(const fg_batch* b, std::vector<double>& p) {
  const size_t n = b->g.size(); p.assign(n, 0.0); double tot = 0.0;
  for (size_t j = 0; j < n; ++j) { const double C = per_sample_sigma(b->g[j].sum); p[j] = C / std::sqrt(b->g[j].t > 0.0 ? b->g[j].t : 1.0); tot = tot + p[j]; }
  if (!(tot > 0.0)) { for (size_t j = 0; j < n; ++j) p[j] = 1.0 / (double)n; return; }   // nothing known yet: uniform
  for (size_t j = 0; j < n; ++j) p[j] = p[j] / tot;
}

extern "C" {

int fg_batch_create(fg_plan* const* plans, int32_t n_plans, fg_batch** out) {
  if (!out) return bfail(FG_E_ARG, "out is NULL");
  *out = nullptr;
  if (!plans || n_plans <= 0) return bfail(FG_E_ARG, "no plans");
  fg_batch* b = new fg_batch();
  for (int j = 0; j < n_plans; ++j) { if (!plans[j]) { delete b; return bfail(FG_E_ARG, "NULL plan"); } GraphState s; s.plan = plans[j]; std::memset(&s.sum, 0, sizeof(s.sum)); b->g.push_back(s); }
  *out = b; return FG_OK;
}
void fg_batch_destroy(fg_batch* b) { delete b; }

int fg_batch_set_times(fg_batch* b, const double* seconds_per_sample) {
  if (!b || !seconds_per_sample) return bfail(FG_E_ARG, "NULL argument");
  for (size_t j = 0; j < b->g.size(); ++j) { if (!(seconds_per_sample[j] > 0.0)) return bfail(FG_E_ARG, "times must be > 0"); b->g[j].t = seconds_per_sample[j]; }
  return FG_OK;
}

int fg_batch_fold(fg_batch* b, int32_t j, const fg_result* r, double seconds) {
  if (!b || !r || j < 0 || j >= (int)b->g.size()) return bfail(FG_E_ARG, "bad argument");
  GraphState& s = b->g[j];
  if (!s.has) { s.sum = *r; s.has = true; }
  else { fg_result m; int rc = fg_result_merge(&s.sum, r, &m); if (rc != FG_OK) return rc; s.sum = m; }
  if (seconds > 0.0 && r->n_samples > 0) s.t = seconds / (double)r->n_samples;      // latest measurement of t_j
  update_tolerances(b);
  return FG_OK;
}

int fg_batch_pilot(fg_batch* b, uint64_t n_pilot, uint64_t seed, uint64_t first_sample, double target_samples, double rel_tol, void* stream) {
  if (!b || n_pilot == 0) return bfail(FG_E_ARG, "bad argument");
  if (!(rel_tol >= 0.0) || !(target_samples >= 0.0)) return bfail(FG_E_ARG, "bad tolerance / target");
  b->rel_tol = rel_tol; b->target = target_samples;
  for (size_t j = 0; j < b->g.size(); ++j) {
    GraphState& s = b->g[j];
    // the initialisation stage has no sigma yet: a loose relative criterion keeps the precision ladder working
    int rc = fg_plan_set_tol(s.plan, 1e-6, 0.0); if (rc != FG_OK) return rc;
    rc = fg_plan_profile(s.plan, 1); if (rc != FG_OK) return rc;
    fg_result r; rc = fg_integrate_range(s.plan, first_sample, n_pilot, seed, stream, &r); if (rc != FG_OK) return rc;
    double ms[3] = {0, 0, 0}; int64_t nl = 0; rc = fg_plan_timing(s.plan, ms, &nl); if (rc != FG_OK) return rc;
    fg_plan_profile(s.plan, 0);
    s.next_sample = first_sample + n_pilot;
    rc = fg_batch_fold(b, (int32_t)j, &r, (ms[0] + ms[1] + ms[2]) * 1e-3); if (rc != FG_OK) return rc;
  }
  for (auto& s : b->g) {
    const bool both0 = b->rel_tol == 0.0 && s.abs_tol == 0.0;        // a graph with zero measured variance
    int rc = fg_plan_set_tol(s.plan, both0 ? 1e-12 : b->rel_tol, s.abs_tol); if (rc != FG_OK) return rc;
  }
  return FG_OK;
}

int fg_batch_probabilities(const fg_batch* b, double* p) {
  if (!b || !p) return bfail(FG_E_ARG, "NULL argument");
  std::vector<double> v; probabilities(b, v);
  for (size_t j = 0; j < v.size(); ++j) p[j] = v[j];
  return FG_OK;
}

int fg_batch_next(fg_batch* b, uint64_t sched_seed, uint64_t block_samples, int32_t* graph, uint64_t* first_sample) {
  if (!b || !graph || !first_sample || block_samples == 0) return bfail(FG_E_ARG, "bad argument");
  std::vector<double> p; probabilities(b, p);
  uint32_t w[4]; const uint64_t k = b->blocks_drawn++;
  philox4x32_10((uint32_t)k, (uint32_t)(k >> 32), 0u, 0u, (uint32_t)sched_seed, (uint32_t)(sched_seed >> 32), w);
  const double u = uniform53(w[0], w[1]);
  double cum = 0.0; int pick = (int)p.size() - 1;
  for (size_t j = 0; j < p.size(); ++j) { cum = cum + p[j]; if (u < cum) { pick = (int)j; break; } }
  *graph = pick; *first_sample = b->g[pick].next_sample; b->g[pick].next_sample += block_samples;
  return FG_OK;
}

int fg_batch_run(fg_batch* b, uint64_t n_blocks, uint64_t block_samples, uint64_t seed, uint64_t sched_seed, void* stream) {
  if (!b) return bfail(FG_E_ARG, "NULL batch");
  for (uint64_t k = 0; k < n_blocks; ++k) {
    int32_t j; uint64_t first; int rc = fg_batch_next(b, sched_seed, block_samples, &j, &first); if (rc != FG_OK) return rc;
    GraphState& s = b->g[j];
    const bool both0 = b->rel_tol == 0.0 && s.abs_tol == 0.0;
    rc = fg_plan_set_tol(s.plan, both0 ? 1e-12 : b->rel_tol, s.abs_tol); if (rc != FG_OK) return rc;      // (18) with the current sigmas
    rc = fg_plan_profile(s.plan, 1); if (rc != FG_OK) return rc;
    fg_result r; rc = fg_integrate_range(s.plan, first, block_samples, seed, stream, &r); if (rc != FG_OK) return rc;
    double ms[3] = {0, 0, 0}; int64_t nl = 0; rc = fg_plan_timing(s.plan, ms, &nl); if (rc != FG_OK) return rc;
    fg_plan_profile(s.plan, 0);
    rc = fg_batch_fold(b, j, &r, (ms[0] + ms[1] + ms[2]) * 1e-3); if (rc != FG_OK) return rc;
  }
  return FG_OK;
}

int fg_batch_result(const fg_batch* b, int32_t j, fg_result* out, double* abs_tol, double* seconds_per_sample) {
  if (!b || j < 0 || j >= (int)b->g.size()) return bfail(FG_E_ARG, "bad argument");
  if (out) *out = b->g[j].sum;
  if (abs_tol) *abs_tol = b->g[j].abs_tol;
  if (seconds_per_sample) *seconds_per_sample = b->g[j].t;
  return FG_OK;
}

int fg_batch_total(const fg_batch* b, double* value, double* sigma_down, uint64_t* n_total) {
  if (!b) return bfail(FG_E_ARG, "NULL batch");
  double v = 0.0, s2 = 0.0; uint64_t n = 0;
  for (auto& s : b->g) { v += s.sum.mean; s2 += s.sum.variance > 0.0 ? s.sum.variance : 0.0; n += s.sum.n_samples; }
  if (value) *value = v;
  if (sigma_down) *sigma_down = std::sqrt(s2);     // (19)
  if (n_total) *n_total = n;
  return FG_OK;
}

int fg_batch_set_classes(fg_batch* b, const int32_t* kmm_per_graph) {
  if (!b || !kmm_per_graph) return bfail(FG_E_ARG, "NULL argument");
  for (size_t j = 0; j < b->g.size(); ++j) for (int i = 0; i < 3; ++i) b->g[j].kmm[i] = kmm_per_graph[3 * j + i];
  return FG_OK;
}

int fg_batch_class_total(const fg_batch* b, const int32_t* kmm, double* value, double* sigma_down, int32_t* n_graphs) {
  if (!b || !kmm) return bfail(FG_E_ARG, "NULL argument");
  double v = 0.0, s2 = 0.0; int32_t n = 0;
  for (auto& s : b->g) if (s.kmm[0] == kmm[0] && s.kmm[1] == kmm[1] && s.kmm[2] == kmm[2]) { v += s.sum.mean; s2 += s.sum.variance > 0.0 ? s.sum.variance : 0.0; ++n; }
  if (value) *value = v;
  if (sigma_down) *sigma_down = std::sqrt(s2);     // (19) restricted to the class
  if (n_graphs) *n_graphs = n;
  return FG_OK;
}

}  // extern "C"
