// Owner assignment from a measured execution-cost model (section 3.4).  Host code only.
//
//   minimise   max_r  sum_{s,b} c[s,b] x[s,b,r]
//   subject to sum_{r,b} b x[s,b,r] = n_s  for every shape s,   x integer >= 0            (Eq. 5, PAPER.md:199-202;
//                                                                 the "Z_{>0}" printed there must be Z_{>=0})
//
// c[s,b] = measured time of one batch of b matrices of shape s (dmuon_measure_cost).  The paper solves the MILP with
// SciPy below a search-space threshold and falls back to a greedy search above it.  Here the
// exact solver is a depth-first branch and bound (small instances: tests, few shapes), the greedy one is longest-
// processing-time-first over several batch-size caps.  Output layout: x[(k * R) + r] with k the running index of
// (s, b) in the concatenated batch-size lists.
#include <algorithm>
#include <cmath>
#include <limits>
#include <numeric>

#include "planner.h"

namespace dmuon {
namespace {

struct Config {       // one (s, b)
  int shape, b, k;
  double c;
};

std::vector<std::vector<Config>> configs_of(const AssignInput& in) {
  std::vector<std::vector<Config>> out(in.num_shapes);
  int k = 0;
  for (int s = 0; s < in.num_shapes; ++s)
    for (int j = 0; j < in.num_batches[s]; ++j, ++k) out[s].push_back(Config{s, in.batch_sizes[k], k, in.costs[k]});
  return out;
}

// Cheapest way to cut n matrices of one shape into batches of the allowed sizes <= cap (unbounded knapsack, exact sum).
// Returns false if n cannot be formed.
bool decompose(const std::vector<Config>& cfgs, int n, int cap, std::vector<const Config*>* jobs) {
  const double inf = std::numeric_limits<double>::infinity();
  std::vector<double> best(n + 1, inf);
  std::vector<const Config*> via(n + 1, nullptr);
  best[0] = 0.0;
  for (int v = 1; v <= n; ++v)
    for (const Config& c : cfgs)
      if (c.b <= cap && c.b <= v && best[v - c.b] + c.c < best[v]) { best[v] = best[v - c.b] + c.c; via[v] = &c; }
  if (n > 0 && !via[n]) return false;
  for (int v = n; v > 0; v -= via[v]->b) jobs->push_back(via[v]);
  return true;
}

}  // namespace

int assign_owners_greedy(const AssignInput& in, int32_t* x_out, double* makespan) {
  const int R = in.num_ranks;
  const auto cfgs = configs_of(in);
  int total_k = 0;
  for (int s = 0; s < in.num_shapes; ++s) total_k += in.num_batches[s];
  std::vector<int> caps;
  for (const auto& v : cfgs) for (const Config& c : v) caps.push_back(c.b);
  std::sort(caps.begin(), caps.end(), std::greater<int>());
  caps.erase(std::unique(caps.begin(), caps.end()), caps.end());
  if (caps.empty()) caps.push_back(1);
  double best_ms = std::numeric_limits<double>::infinity();
  std::vector<int32_t> best_x(static_cast<size_t>(total_k) * R, 0);
  for (int cap : caps) {
    std::vector<const Config*> jobs;
    bool ok = true;
    for (int s = 0; s < in.num_shapes && ok; ++s) ok = decompose(cfgs[s], in.counts[s], cap, &jobs);
    if (!ok) continue;
    // longest processing time first onto the least-loaded rank
    std::stable_sort(jobs.begin(), jobs.end(), [](const Config* a, const Config* b) { return a->c > b->c; });
    std::vector<double> load(R, 0.0);
    std::vector<int32_t> x(static_cast<size_t>(total_k) * R, 0);
    for (const Config* j : jobs) {
      const int r = static_cast<int>(std::min_element(load.begin(), load.end()) - load.begin());
      load[r] += j->c;
      x[static_cast<size_t>(j->k) * R + r] += 1;
    }
    const double ms = *std::max_element(load.begin(), load.end());
    if (ms < best_ms) { best_ms = ms; best_x = x; }
  }
  if (!std::isfinite(best_ms)) {
    if (std::accumulate(in.counts, in.counts + in.num_shapes, 0LL) == 0) best_ms = 0.0;
    else { set_error("dmuon_assign_owners: a shape's count cannot be formed from its batch sizes"); return DMUON_ERR_INVALID_ARG; }
  }
  std::copy(best_x.begin(), best_x.end(), x_out);
  *makespan = best_ms;
  return DMUON_OK;
}

namespace {

struct Search {
  const AssignInput* in;
  std::vector<std::vector<Config>> cfgs;   // per shape, sorted by batch size descending
  int R;
  std::vector<int> remaining;
  std::vector<double> load;
  std::vector<int32_t> x, best_x;
  double best;
  long long nodes, limit;
  bool aborted;

  // lower bound: the cheapest possible cost per matrix of each shape, spread perfectly
  double bound() const {
    double rest = 0.0;
    for (size_t s = 0; s < cfgs.size(); ++s) {
      if (!remaining[s]) continue;
      double per = std::numeric_limits<double>::infinity();
      for (const Config& c : cfgs[s]) per = std::min(per, c.c / c.b);
      rest += per * remaining[s];
    }
    const double total = std::accumulate(load.begin(), load.end(), 0.0) + rest;
    return std::max(total / R, *std::max_element(load.begin(), load.end()));
  }

  // place batches of shape s: batch sizes in non-increasing order (first index into cfgs[s] allowed: `from`), and for
  // equal consecutive batch sizes ranks in non-decreasing order (`rank_from`), which removes permutations of equal jobs
  void go(int s, size_t from, int rank_from) {
    if (aborted) return;
    if (++nodes > limit) { aborted = true; return; }
    while (s < static_cast<int>(cfgs.size()) && remaining[s] == 0) { ++s; from = 0; rank_from = 0; }
    if (s == static_cast<int>(cfgs.size())) {
      const double ms = *std::max_element(load.begin(), load.end());
      if (ms < best) { best = ms; best_x = x; }
      return;
    }
    if (bound() >= best) return;
    for (size_t j = from; j < cfgs[s].size(); ++j) {
      const Config& c = cfgs[s][j];
      if (c.b > remaining[s]) continue;
      for (int r = (j == from ? rank_from : 0); r < R; ++r) {
        // ranks with identical loads AND identical assignments so far are interchangeable: try only the first empty one
        bool dup = false;
        if (load[r] == 0.0)
          for (int q = 0; q < r && !dup; ++q) dup = load[q] == 0.0;
        if (dup) continue;
        if (load[r] + c.c >= best) continue;
        load[r] += c.c;
        remaining[s] -= c.b;
        x[static_cast<size_t>(c.k) * R + r] += 1;
        go(s, j, r);
        x[static_cast<size_t>(c.k) * R + r] -= 1;
        remaining[s] += c.b;
        load[r] -= c.c;
      }
    }
  }
};

}  // namespace

int assign_owners_exact(const AssignInput& in, int32_t* x_out, double* makespan, long long node_limit) {
  Search S;
  S.in = &in;
  S.cfgs = configs_of(in);
  for (auto& v : S.cfgs) std::stable_sort(v.begin(), v.end(), [](const Config& a, const Config& b) { return a.b > b.b; });
  S.R = in.num_ranks;
  S.remaining.assign(in.counts, in.counts + in.num_shapes);
  S.load.assign(S.R, 0.0);
  int total_k = 0;
  for (int s = 0; s < in.num_shapes; ++s) total_k += in.num_batches[s];
  S.x.assign(static_cast<size_t>(total_k) * S.R, 0);
  // start from the greedy solution: a good incumbent prunes most of the tree
  std::vector<int32_t> gx(S.x.size(), 0);
  double gms = 0.0;
  int rc = assign_owners_greedy(in, gx.data(), &gms);
  if (rc) return rc;
  S.best = gms * (1.0 + 1e-12) + 1e-300;
  S.best_x = gx;
  S.nodes = 0;
  S.limit = node_limit;
  S.aborted = false;
  S.go(0, 0, 0);
  if (S.aborted) { set_error("dmuon_assign_owners: exact search exceeded %lld nodes", node_limit); return DMUON_ERR_INTERNAL; }
  std::copy(S.best_x.begin(), S.best_x.end(), x_out);
  double ms = 0.0;
  {
    std::vector<double> load(S.R, 0.0);
    int k = 0;
    for (int s = 0; s < in.num_shapes; ++s)
      for (int j = 0; j < in.num_batches[s]; ++j, ++k)
        for (int r = 0; r < S.R; ++r) load[r] += in.costs[k] * S.best_x[static_cast<size_t>(k) * S.R + r];
    ms = *std::max_element(load.begin(), load.end());
  }
  *makespan = ms;
  return DMUON_OK;
}

}  // namespace dmuon
