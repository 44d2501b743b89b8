// C ABI of libdmuon (include/dmuon.h): argument validation, options, error strings, profiling events, and the
// enqueue order of the Muon step:  momentum+Nesterov+cast+sumsq -> norms -> normalise/orient/cast -> k x (SYRK, SQ, BX)
// per shape bucket -> apply.   (Eq. 1, Eq. 2, Alg. 1 l.12-15.)
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>

#include "planner.h"

namespace dmuon {

namespace {

thread_local char g_err[512] = "";
Options g_opt;
Plan* g_last_plan = nullptr;     // plan of the most recent step / ns call (for dmuon_read_ns_output)
void* g_ext_ws = nullptr;
size_t g_ext_ws_bytes = 0;

// ---------------------------------------------------------------- profiling
struct ProfRec {
  std::string name;
  cudaEvent_t e0, e1;
};
std::vector<ProfRec> g_prof_open;                 // recorded, not yet folded
std::vector<cudaEvent_t> g_event_pool;
std::map<std::string, std::pair<long long, double>> g_prof_acc;   // name -> (launches, ms)
long long g_launches = 0;

cudaEvent_t take_event() {
  if (!g_event_pool.empty()) {
    cudaEvent_t e = g_event_pool.back();
    g_event_pool.pop_back();
    return e;
  }
  cudaEvent_t e = nullptr;
  cudaEventCreate(&e);
  return e;
}

int fold_profile() {
  for (ProfRec& r : g_prof_open) {
    if (cudaEventSynchronize(r.e1) != cudaSuccess) { cudaGetLastError(); set_error("profile: event sync failed"); return DMUON_ERR_CUDA; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, r.e0, r.e1);
    auto& acc = g_prof_acc[r.name];
    acc.first += 1;
    acc.second += ms;
    g_event_pool.push_back(r.e0);
    g_event_pool.push_back(r.e1);
  }
  g_prof_open.clear();
  return DMUON_OK;
}

int validate(const void* const* a, const void* const* b, const void* const* c, const int32_t* shapes, int32_t count,
             const char* fn) {
  if (count < 0) { set_error("%s: count < 0", fn); return DMUON_ERR_INVALID_ARG; }
  if (count == 0) return DMUON_OK;
  if (!a || !shapes) { set_error("%s: null argument", fn); return DMUON_ERR_INVALID_ARG; }
  for (int i = 0; i < count; ++i) {
    if (shapes[2 * i] <= 0 || shapes[2 * i + 1] <= 0) {
      set_error("%s: matrix %d has non-positive dimension %d x %d", fn, i, shapes[2 * i], shapes[2 * i + 1]);
      return DMUON_ERR_INVALID_ARG;
    }
    const void* ptrs[3] = {a[i], b ? b[i] : a[i], c ? c[i] : a[i]};
    for (const void* p : ptrs) {
      if (!p) { set_error("%s: matrix %d has a null pointer", fn, i); return DMUON_ERR_INVALID_ARG; }
      if (reinterpret_cast<uintptr_t>(p) & 15) { set_error("%s: matrix %d pointer %p is not 16-byte aligned", fn, i, p); return DMUON_ERR_INVALID_ARG; }
    }
  }
  return DMUON_OK;
}

// Patch the per-call pointers into the plan's records and upload them if anything changed.
int bind_pointers(Plan& plan, void* const* w, const void* const* g, void* const* m, int steps, const float* coeffs,
                  bool per_step, cudaStream_t stream, void* const* masters = nullptr) {
  const int count = static_cast<int>(plan.mats.size());
  bool dirty = false;
  std::vector<int> parity(plan.buckets.size());
  for (size_t b = 0; b < plan.buckets.size(); ++b)
    parity[b] = result_parity(plan, plan.buckets[b], steps, coeffs, per_step, g_opt);
  for (int i = 0; i < count; ++i) {
    MatRec& r = plan.h_recs[i];
    void* gi = g ? const_cast<void*>(g[i]) : nullptr;
    void* mi = m ? m[i] : nullptr;
    float* w32 = masters ? static_cast<float*>(masters[i]) : nullptr;
    if (r.W != w[i] || r.G != gi || r.M != mi || r.W32 != w32) dirty = true;
    r.W32 = w32;
    r.W = w[i];
    r.G = gi;
    r.M = mi;
    const MatrixInfo& info = plan.mats[i];
    const void* o = plan.ws + (parity[info.bucket] ? info.off_p : info.off_q);   // X0 in Q; each block swaps buffers
    if (r.O != o) dirty = true;
    r.O = o;
  }
  if (dirty && count > 0)
    DMUON_CUDA_CHECK(cudaMemcpyAsync(plan.d_recs, plan.h_recs.data(), sizeof(MatRec) * count, cudaMemcpyHostToDevice, stream));
  return DMUON_OK;
}

int muon_step_device(void* const* params, const void* const* grads, void* const* momenta, const int32_t* shapes,
                     int32_t count, float lr, float mu, float wd, cudaStream_t stream, Plan** plan_out,
                     void* const* masters = nullptr) {
  Plan* plan = nullptr;
  int rc = get_plan(shapes, count, g_opt, g_ext_ws, g_ext_ws_bytes, stream, &plan);
  if (rc) return rc;
  if (plan_out) *plan_out = plan;
  g_last_plan = plan;
  if ((rc = bind_pointers(*plan, params, grads, momenta, g_opt.steps, g_opt.coeffs, false, stream, masters))) return rc;
  const bool master = masters != nullptr;
  if (plan->parts.empty() || !g_opt.overlap) {
    const ElemTables& T = plan->tables;
    if ((rc = launch_momentum(T, mu, stream))) return rc;
    if ((rc = launch_finalize_norms(T, g_opt.eps, stream))) return rc;
    if ((rc = launch_normalize(T, /*from_user=*/false, plan->fp32, stream))) return rc;
    if ((rc = run_ns_steps(*plan, g_opt.steps, g_opt.coeffs, false, g_opt, stream))) return rc;
    if ((rc = launch_apply(T, lr, wd, plan->fp32, master, stream))) return rc;
    return DMUON_OK;
  }
  // Several buckets: the HBM-bound passes of one bucket run on the plan's side stream under the GEMMs of another.
  //   main:  prep(part 0) | NS(bucket 0) | NS(bucket 1) | ... | NS(last) | apply(last) | join
  //   side:  prep(parts 1..)             | apply(part 0) after NS(bucket 0) | apply(part 1) after NS(bucket 1) | ...
  // prep = momentum + norms + normalise.  Matrices of different buckets share no buffer, so only the fork/join and the
  // per-bucket "ready" / "NS done" events order the two streams.
  const int nb = static_cast<int>(plan->parts.size());
  cudaStream_t side = plan->side;
  cudaEvent_t ev_fork = plan->ev[2 * nb], ev_join = plan->ev[2 * nb + 1];
  auto prep = [&](const ElemTables& T, cudaStream_t s) -> int {
    int r;
    if ((r = launch_momentum(T, mu, s))) return r;
    if ((r = launch_finalize_norms(T, g_opt.eps, s))) return r;
    return launch_normalize(T, /*from_user=*/false, false, s);
  };
  DMUON_CUDA_CHECK(cudaEventRecord(ev_fork, stream));            // after the pointer upload and the caller's earlier work
  DMUON_CUDA_CHECK(cudaStreamWaitEvent(side, ev_fork, 0));
  if ((rc = prep(plan->parts[0], stream))) return rc;
  for (int k = 1; k < nb; ++k) {
    if ((rc = prep(plan->parts[k], side))) return rc;
    DMUON_CUDA_CHECK(cudaEventRecord(plan->ev[2 * k], side));   // bucket k's X0 is ready
  }
  for (int k = 0; k < nb; ++k) {
    if (k > 0) DMUON_CUDA_CHECK(cudaStreamWaitEvent(stream, plan->ev[2 * k], 0));
    if ((rc = run_ns_bucket(*plan, plan->order[k], g_opt.steps, g_opt.coeffs, false, g_opt, stream))) return rc;
    if (k + 1 < nb) {
      DMUON_CUDA_CHECK(cudaEventRecord(plan->ev[2 * k + 1], stream));                 // bucket k's O is ready
      DMUON_CUDA_CHECK(cudaStreamWaitEvent(side, plan->ev[2 * k + 1], 0));
      if ((rc = launch_apply(plan->parts[k], lr, wd, false, master, side))) return rc;
    } else {
      if ((rc = launch_apply(plan->parts[k], lr, wd, false, master, stream))) return rc;
    }
  }
  DMUON_CUDA_CHECK(cudaEventRecord(ev_join, side));
  DMUON_CUDA_CHECK(cudaStreamWaitEvent(stream, ev_join, 0));
  return DMUON_OK;
}

int ns_batched_impl(void* const* ptrs, const int32_t* shapes, int32_t count, int32_t steps, const float* coeffs,
                    bool per_step, cudaStream_t stream) {
  static const float kDefault[3] = {3.4445f, -4.7750f, 2.0315f};
  if (steps < 0) { set_error("dmuon_ns_batched: steps < 0"); return DMUON_ERR_INVALID_ARG; }
  int rc = validate(reinterpret_cast<const void* const*>(ptrs), nullptr, nullptr, shapes, count, "dmuon_ns_batched");
  if (rc || count == 0) return rc;
  if (!coeffs) {
    if (per_step && steps > 0) { set_error("dmuon_ns_batched_sched: coeffs is null"); return DMUON_ERR_INVALID_ARG; }
    coeffs = kDefault;
    per_step = false;
  }
  Plan* plan = nullptr;
  if ((rc = get_plan(shapes, count, g_opt, g_ext_ws, g_ext_ws_bytes, stream, &plan))) return rc;
  g_last_plan = plan;
  if ((rc = bind_pointers(*plan, ptrs, nullptr, nullptr, steps, coeffs, per_step, stream))) return rc;
  const ElemTables& T = plan->tables;
  if ((rc = launch_sumsq(T, stream))) return rc;
  if ((rc = launch_finalize_norms(T, g_opt.eps, stream))) return rc;
  if ((rc = launch_normalize(T, /*from_user=*/true, plan->fp32, stream))) return rc;
  if ((rc = run_ns_steps(*plan, steps, coeffs, per_step, g_opt, stream))) return rc;
  if ((rc = launch_store_ns(T, plan->fp32, stream))) return rc;
  return DMUON_OK;
}

// ---- state of dmuon_muon_step_host: device staging of W | G | M, copy streams, events (one shape set at a time)
struct HostCtx {
  std::vector<int32_t> shapes;
  uint8_t* stage = nullptr;
  std::vector<size_t> off;      // per matrix offset of W; G at + third, M at + 2 * third
  size_t third = 0;
  int group = 0;                // matrices per group
  cudaStream_t s_in = nullptr, s_out = nullptr;
  std::vector<cudaEvent_t> ev;  // [2 g] copy-in done, [2 g + 1] step done, then start / end
  int release() {
    if (stage || s_in) cudaDeviceSynchronize();
    if (stage) cudaFree(stage);
    if (s_in) cudaStreamDestroy(s_in);
    if (s_out) cudaStreamDestroy(s_out);
    for (cudaEvent_t e : ev) cudaEventDestroy(e);
    cudaGetLastError();
    *this = HostCtx();
    return DMUON_OK;
  }
} g_host;

// ---- dmuon_ns_gemm table cache (one entry: the last argument set)
struct GemmCall {
  std::vector<const void*> in0, in1;
  std::vector<void*> out;
  int op = -1, m = 0, n = 0, variant = -2;
  GemmProblem* d_probs = nullptr;
  TileUnit* d_units = nullptr;
  int units = 0;
} g_gemm_call;

}  // namespace

void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof g_err, fmt, ap);
  va_end(ap);
}

void prof_begin(const char* name, cudaStream_t s) {
  ++g_launches;
  if (!g_opt.profile) return;
  ProfRec r{name, take_event(), take_event()};
  cudaEventRecord(r.e0, s);
  g_prof_open.push_back(r);
}

void prof_end(cudaStream_t s) {
  if (!g_opt.profile || g_prof_open.empty()) return;
  cudaEventRecord(g_prof_open.back().e1, s);
}

}  // namespace dmuon

using namespace dmuon;

extern "C" {

DMUON_API const char* dmuon_version(void) { return "libdmuon 0.1 (sm_100a)"; }

DMUON_API const char* dmuon_last_error(void) { return g_err; }

DMUON_API int dmuon_set_option(const char* key, const char* value) {
  if (!key || !value) { set_error("dmuon_set_option: null argument"); return DMUON_ERR_INVALID_ARG; }
  const std::string k(key), v(value);
  auto as_bool = [&](bool* out) {
    if (v == "1" || v == "true" || v == "on") { *out = true; return true; }
    if (v == "0" || v == "false" || v == "off") { *out = false; return true; }
    return false;
  };
  if (k == "steps") {
    char* end = nullptr;
    long s = strtol(value, &end, 10);
    if (end == value || *end || s < 0 || s > 64) { set_error("option steps: bad value '%s'", value); return DMUON_ERR_INVALID_ARG; }
    g_opt.steps = static_cast<int>(s);
    return DMUON_OK;
  }
  if (k == "coeffs") {
    float a, b, c;
    char tail;
    if (sscanf(value, " %f , %f , %f %c", &a, &b, &c, &tail) != 3) { set_error("option coeffs: expected 'a,b,c', got '%s'", value); return DMUON_ERR_INVALID_ARG; }
    g_opt.coeffs[0] = a; g_opt.coeffs[1] = b; g_opt.coeffs[2] = c;
    return DMUON_OK;
  }
  if (k == "mode") {
    if (v == "tc") g_opt.fp32_check = false;
    else if (v == "fp32_check") g_opt.fp32_check = true;
    else { set_error("option mode: expected 'tc' or 'fp32_check', got '%s'", value); return DMUON_ERR_INVALID_ARG; }
    return DMUON_OK;
  }
  if (k == "autotune") { if (as_bool(&g_opt.autotune)) return DMUON_OK; set_error("option autotune: bad value '%s'", value); return DMUON_ERR_INVALID_ARG; }
  if (k == "profile") { if (as_bool(&g_opt.profile)) return DMUON_OK; set_error("option profile: bad value '%s'", value); return DMUON_ERR_INVALID_ARG; }
  if (k == "schedule") {
    if (v == "auto") g_opt.gram_blocks = true;
    else if (v == "x") g_opt.gram_blocks = false;
    else { set_error("option schedule: expected 'auto' or 'x', got '%s'", value); return DMUON_ERR_INVALID_ARG; }
    return DMUON_OK;
  }
  if (k == "variants") {
    int a, b, c;
    char tail;
    if (sscanf(value, " %d , %d , %d %c", &a, &b, &c, &tail) != 3 || a < -1 || b < -1 || c < -1 || a >= kNumVariants ||
        b >= kNumVariants || c >= kNumVariants) { set_error("option variants: expected 'syrk,sq,bx' in -1..%d, got '%s'", kNumVariants - 1, value); return DMUON_ERR_INVALID_ARG; }
    g_opt.force_variant[0] = a; g_opt.force_variant[1] = b; g_opt.force_variant[2] = c;
    return DMUON_OK;
  }
  if (k == "overlap") { if (as_bool(&g_opt.overlap)) return DMUON_OK; set_error("option overlap: bad value '%s'", value); return DMUON_ERR_INVALID_ARG; }
  if (k == "cache_path") { g_opt.cache_path = v; g_opt.cache_path_set = true; return DMUON_OK; }
  set_error("dmuon_set_option: unknown key '%s'", key);
  return DMUON_ERR_INVALID_ARG;
}

DMUON_API int dmuon_ns_batched(void* const* ptrs, const int32_t* shapes, int32_t count, int32_t steps,
                               const float* coeffs, dmuon_stream_t stream) {
  return ns_batched_impl(ptrs, shapes, count, steps, coeffs, false, reinterpret_cast<cudaStream_t>(stream));
}

DMUON_API int dmuon_ns_batched_sched(void* const* ptrs, const int32_t* shapes, int32_t count, int32_t steps,
                                     const float* coeffs, dmuon_stream_t stream) {
  return ns_batched_impl(ptrs, shapes, count, steps, coeffs, true, reinterpret_cast<cudaStream_t>(stream));
}

DMUON_API int dmuon_muon_step(void* const* params, const void* const* grads, void* const* momenta,
                              const int32_t* shapes, int32_t count, float lr, float mu, float wd,
                              dmuon_stream_t stream) {
  int rc = validate(reinterpret_cast<const void* const*>(params), grads, reinterpret_cast<const void* const*>(momenta),
                    shapes, count, "dmuon_muon_step");
  if (rc || count == 0) return rc;
  if (!grads || !momenta) { set_error("dmuon_muon_step: null argument"); return DMUON_ERR_INVALID_ARG; }
  return muon_step_device(params, grads, momenta, shapes, count, lr, mu, wd, reinterpret_cast<cudaStream_t>(stream), nullptr);
}

DMUON_API int dmuon_muon_step_master(void* const* params, void* const* masters, const void* const* grads,
                                     void* const* momenta, const int32_t* shapes, int32_t count, float lr, float mu,
                                     float wd, dmuon_stream_t stream) {
  int rc = validate(reinterpret_cast<const void* const*>(params), grads, reinterpret_cast<const void* const*>(momenta),
                    shapes, count, "dmuon_muon_step_master");
  if (rc || count == 0) return rc;
  if (!grads || !momenta || !masters) { set_error("dmuon_muon_step_master: null argument"); return DMUON_ERR_INVALID_ARG; }
  for (int i = 0; i < count; ++i) {
    if (!masters[i]) { set_error("dmuon_muon_step_master: matrix %d has a null master pointer", i); return DMUON_ERR_INVALID_ARG; }
    if (reinterpret_cast<uintptr_t>(masters[i]) & 31) { set_error("dmuon_muon_step_master: master %d (%p) is not 32-byte aligned", i, masters[i]); return DMUON_ERR_INVALID_ARG; }
  }
  return muon_step_device(params, grads, momenta, shapes, count, lr, mu, wd, reinterpret_cast<cudaStream_t>(stream), nullptr, masters);
}

// Host-buffer entry: the matrix list is cut into groups of whole periods of its shape pattern (a transformer's layers),
// so that every group has the same shape list and shares one plan and one workspace.  Group g's host->device copies
// (copy-in stream), the step of group g-1 (caller's stream) and the device->host copies of group g-2 (copy-out stream)
// overlap; PCIe carries both directions at once.
DMUON_API int dmuon_muon_step_host(void* const* params_host, const void* const* grads_host, void* const* momenta_host,
                                   const int32_t* shapes, int32_t count, float lr, float mu, float wd,
                                   dmuon_stream_t stream_) {
  cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
  if (count < 0) { set_error("dmuon_muon_step_host: count < 0"); return DMUON_ERR_INVALID_ARG; }
  if (count == 0) return DMUON_OK;
  if (!params_host || !grads_host || !momenta_host || !shapes) { set_error("dmuon_muon_step_host: null argument"); return DMUON_ERR_INVALID_ARG; }
  for (int i = 0; i < count; ++i) {
    if (shapes[2 * i] <= 0 || shapes[2 * i + 1] <= 0) { set_error("dmuon_muon_step_host: bad shape of matrix %d", i); return DMUON_ERR_INVALID_ARG; }
    if (!params_host[i] || !grads_host[i] || !momenta_host[i]) { set_error("dmuon_muon_step_host: matrix %d has a null pointer", i); return DMUON_ERR_INVALID_ARG; }
  }
  int rc = check_device();
  if (rc) return rc;
  HostCtx& hc = g_host;
  if (hc.shapes.size() != static_cast<size_t>(2 * count) || memcmp(hc.shapes.data(), shapes, sizeof(int32_t) * 2 * count) != 0) {
    if ((rc = hc.release())) return rc;
    hc.shapes.assign(shapes, shapes + 2 * count);
    // smallest period of the shape pattern, then the smallest number of periods per group that gives <= 8 groups
    int period = count;
    for (int p = 1; p < count; ++p) {
      if (count % p) continue;
      bool ok = true;
      for (int k = p; k < count && ok; ++k) ok = shapes[2 * k] == shapes[2 * (k - p)] && shapes[2 * k + 1] == shapes[2 * (k - p) + 1];
      if (ok) { period = p; break; }
    }
    const int periods = count / period;
    int per_group = periods;
    for (int d = 1; d <= periods; ++d)
      if (periods % d == 0 && periods / d <= 8) { per_group = d; break; }
    hc.group = per_group * period;
    size_t off = 0;
    hc.off.resize(count);
    for (int i = 0; i < count; ++i) {
      hc.off[i] = off;
      off += (static_cast<size_t>(shapes[2 * i]) * shapes[2 * i + 1] * 2 + 255) / 256 * 256;
    }
    hc.third = off;
    void* p = nullptr;
    cudaError_t e = cudaMalloc(&p, 3 * off);
    if (e != cudaSuccess) { cudaGetLastError(); hc.shapes.clear(); set_error("staging allocation of %zu bytes failed", 3 * off); return DMUON_ERR_OOM; }
    hc.stage = static_cast<uint8_t*>(p);
    DMUON_CUDA_CHECK(cudaStreamCreateWithFlags(&hc.s_in, cudaStreamNonBlocking));
    DMUON_CUDA_CHECK(cudaStreamCreateWithFlags(&hc.s_out, cudaStreamNonBlocking));
    const int groups = count / hc.group;
    hc.ev.resize(2 * groups + 2);
    for (cudaEvent_t& ev : hc.ev) DMUON_CUDA_CHECK(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
  }
  const int groups = count / hc.group;
  cudaEvent_t ev_start = hc.ev[2 * groups], ev_end = hc.ev[2 * groups + 1];
  DMUON_CUDA_CHECK(cudaEventRecord(ev_start, stream));            // copies start after the caller's earlier work
  DMUON_CUDA_CHECK(cudaStreamWaitEvent(hc.s_in, ev_start, 0));
  std::vector<void*> w(count), m(count);
  std::vector<const void*> g(count);
  auto bytes_of = [&](int i) { return static_cast<size_t>(shapes[2 * i]) * shapes[2 * i + 1] * 2; };
  for (int i = 0; i < count; ++i) {
    w[i] = hc.stage + hc.off[i];
    g[i] = hc.stage + hc.third + hc.off[i];
    m[i] = hc.stage + 2 * hc.third + hc.off[i];
  }
  g_launches += 5 * count;                                         // 3 H2D + 2 D2H copies per matrix
  for (int gi = 0; gi < groups; ++gi) {
    const int b = gi * hc.group, e = b + hc.group;
    for (int i = b; i < e; ++i) {
      DMUON_CUDA_CHECK(cudaMemcpyAsync(w[i], params_host[i], bytes_of(i), cudaMemcpyHostToDevice, hc.s_in));
      DMUON_CUDA_CHECK(cudaMemcpyAsync(const_cast<void*>(g[i]), grads_host[i], bytes_of(i), cudaMemcpyHostToDevice, hc.s_in));
      DMUON_CUDA_CHECK(cudaMemcpyAsync(m[i], momenta_host[i], bytes_of(i), cudaMemcpyHostToDevice, hc.s_in));
    }
    DMUON_CUDA_CHECK(cudaEventRecord(hc.ev[2 * gi], hc.s_in));
    DMUON_CUDA_CHECK(cudaStreamWaitEvent(stream, hc.ev[2 * gi], 0));
    if ((rc = muon_step_device(w.data() + b, g.data() + b, m.data() + b, shapes + 2 * b, hc.group, lr, mu, wd, stream, nullptr))) return rc;
    DMUON_CUDA_CHECK(cudaEventRecord(hc.ev[2 * gi + 1], stream));
    DMUON_CUDA_CHECK(cudaStreamWaitEvent(hc.s_out, hc.ev[2 * gi + 1], 0));
    for (int i = b; i < e; ++i) {
      DMUON_CUDA_CHECK(cudaMemcpyAsync(params_host[i], w[i], bytes_of(i), cudaMemcpyDeviceToHost, hc.s_out));
      DMUON_CUDA_CHECK(cudaMemcpyAsync(momenta_host[i], m[i], bytes_of(i), cudaMemcpyDeviceToHost, hc.s_out));
    }
  }
  DMUON_CUDA_CHECK(cudaEventRecord(ev_end, hc.s_out));
  DMUON_CUDA_CHECK(cudaStreamWaitEvent(stream, ev_end, 0));      // the caller's stream sees the results
  return DMUON_OK;
}

DMUON_API int dmuon_warmup(const int32_t* shapes, int32_t count, dmuon_stream_t stream) {
  if (count < 0 || (count > 0 && !shapes)) { set_error("dmuon_warmup: bad arguments"); return DMUON_ERR_INVALID_ARG; }
  for (int i = 0; i < count; ++i)
    if (shapes[2 * i] <= 0 || shapes[2 * i + 1] <= 0) { set_error("dmuon_warmup: bad shape of matrix %d", i); return DMUON_ERR_INVALID_ARG; }
  if (count == 0) return DMUON_OK;
  Plan* plan = nullptr;
  return get_plan(shapes, count, g_opt, g_ext_ws, g_ext_ws_bytes, reinterpret_cast<cudaStream_t>(stream), &plan);
}

DMUON_API int dmuon_block_schedule(int32_t rows, int32_t cols, int32_t steps, const float* coeffs, int32_t per_step,
                                   int32_t* out, int32_t cap) {
  if (rows <= 0 || cols <= 0 || steps < 0 || cap < 0 || (cap > 0 && !out) || (per_step && !coeffs && steps > 0)) {
    set_error("dmuon_block_schedule: bad arguments");
    return DMUON_ERR_INVALID_ARG;
  }
  const int m = rows < cols ? rows : cols, n = rows < cols ? cols : rows;
  const int m_pad = (m + kBlk - 1) / kBlk * kBlk, n_pad = (n + kBlk - 1) / kBlk * kBlk;
  const bool gram = g_opt.gram_blocks && gram_eligible(m_pad, n_pad, g_opt.fp32_check);
  const Partition part = choose_partition(steps, coeffs ? coeffs : g_opt.coeffs, coeffs && per_step, gram);
  for (size_t k = 0; k < part.size() && k < static_cast<size_t>(cap); ++k) out[k] = part[k];
  return static_cast<int>(part.size());
}

DMUON_API int dmuon_describe_plan(const int32_t* shapes, int32_t count, int32_t steps, char* buf, size_t len,
                                  dmuon_stream_t stream) {
  if (count < 0 || steps < 0 || (count > 0 && !shapes)) { set_error("dmuon_describe_plan: bad arguments"); return DMUON_ERR_INVALID_ARG; }
  for (int i = 0; i < count; ++i)
    if (shapes[2 * i] <= 0 || shapes[2 * i + 1] <= 0) { set_error("dmuon_describe_plan: bad shape of matrix %d", i); return DMUON_ERR_INVALID_ARG; }
  std::string s = "{\"buckets\": [";
  if (count > 0) {
    Plan* plan = nullptr;
    int rc = get_plan(shapes, count, g_opt, g_ext_ws, g_ext_ws_bytes, reinterpret_cast<cudaStream_t>(stream), &plan);
    if (rc) return rc;
    bool first = true;
    for (const BucketPlan& b : plan->buckets) {
      const Partition part = plan->fp32 ? Partition(steps, 1)
                                        : choose_partition(steps, g_opt.coeffs, false, b.gram && g_opt.gram_blocks);
      char item[160];
      snprintf(item, sizeof item, "%s{\"m\": %d, \"n\": %d, \"count\": %d, \"blocks\": [", first ? "" : ", ", b.m_pad,
               b.n_pad, static_cast<int>(b.mats.size()));
      s += item;
      for (size_t k = 0; k < part.size(); ++k) s += (k ? ", " : "") + std::to_string(part[k]);
      snprintf(item, sizeof item, "], \"variants\": [%d, %d, %d]}", b.variant[0], b.variant[1], b.variant[2]);
      s += item;
      first = false;
    }
  }
  s += "]}";
  if (buf && len > 0) {
    const size_t n = s.size() < len - 1 ? s.size() : len - 1;
    memcpy(buf, s.data(), n);
    buf[n] = 0;
  }
  return static_cast<int>(s.size());
}

DMUON_API size_t dmuon_workspace_bytes(const int32_t* shapes, int32_t count) {
  if (count <= 0 || !shapes) return 0;
  for (int i = 0; i < count; ++i)
    if (shapes[2 * i] <= 0 || shapes[2 * i + 1] <= 0) return 0;
  return plan_workspace_bytes(shapes, count, g_opt.fp32_check);
}

DMUON_API int dmuon_set_workspace(void* dev_ptr, size_t bytes) {
  if ((dev_ptr == nullptr) != (bytes == 0)) { set_error("dmuon_set_workspace: pointer and size must both be set or both be zero"); return DMUON_ERR_INVALID_ARG; }
  if (reinterpret_cast<uintptr_t>(dev_ptr) & 255) { set_error("dmuon_set_workspace: pointer must be 256-byte aligned"); return DMUON_ERR_INVALID_ARG; }
  cudaDeviceSynchronize();
  cudaGetLastError();
  drop_plans();
  g_last_plan = nullptr;
  g_ext_ws = dev_ptr;
  g_ext_ws_bytes = bytes;
  return DMUON_OK;
}

DMUON_API int dmuon_read_ns_output(int32_t index, float* out_dev, dmuon_stream_t stream) {
  if (!g_last_plan) { set_error("dmuon_read_ns_output: no step has run"); return DMUON_ERR_INVALID_ARG; }
  Plan& p = *g_last_plan;
  if (index < 0 || index >= static_cast<int>(p.mats.size()) || !out_dev) { set_error("dmuon_read_ns_output: bad index or null output"); return DMUON_ERR_INVALID_ARG; }
  const MatrixInfo& mi = p.mats[index];
  return launch_export(p.h_recs[index].O, out_dev, mi.rows, mi.cols, mi.n_pad, mi.transposed, p.fp32,
                       reinterpret_cast<cudaStream_t>(stream));
}

DMUON_API int dmuon_profile_reset(void) {
  int rc = fold_profile();
  g_prof_acc.clear();
  g_launches = 0;
  return rc;
}

DMUON_API int dmuon_profile_read(char* buf, size_t len) {
  int rc = fold_profile();
  if (rc) return rc;
  std::string s = "{\"kernels\": {";
  bool first = true;
  for (auto& kv : g_prof_acc) {
    char item[256];
    snprintf(item, sizeof item, "%s\"%s\": {\"launches\": %lld, \"ms\": %.6f}", first ? "" : ", ", kv.first.c_str(),
             kv.second.first, kv.second.second);
    s += item;
    first = false;
  }
  char tail[64];
  snprintf(tail, sizeof tail, "}, \"launches\": %lld}", g_launches);
  s += tail;
  if (buf && len > 0) {
    const size_t n = s.size() < len - 1 ? s.size() : len - 1;
    memcpy(buf, s.data(), n);
    buf[n] = 0;
  }
  return static_cast<int>(s.size());
}

DMUON_API int dmuon_ns_gemm_variants(int32_t op) { return (op >= OP_SYRK && op <= OP_BX) ? kNumVariants : 0; }

DMUON_API int dmuon_ns_gemm(int32_t op, const void* const* in0, const void* const* in1, void* const* out, int32_t m,
                            int32_t n, int32_t count, float alpha, float beta, int32_t variant, dmuon_stream_t stream_) {
  cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
  if (op < 0 || op > 2) { set_error("dmuon_ns_gemm: bad op %d", op); return DMUON_ERR_INVALID_ARG; }
  if (count < 0 || (count > 0 && (!in0 || !out || (op == OP_BX && !in1)))) { set_error("dmuon_ns_gemm: null argument"); return DMUON_ERR_INVALID_ARG; }
  if (op == OP_SQ) n = m;
  if (m <= 0 || n <= 0 || m % kBlk || n % kBlk) { set_error("dmuon_ns_gemm: m and n must be positive multiples of 128 (got %d, %d)", m, n); return DMUON_ERR_INVALID_ARG; }
  if (variant < -1 || (variant >= 0 && !variant_valid(static_cast<GemmOp>(op), variant))) { set_error("dmuon_ns_gemm: variant %d is not defined for op %d", variant, op); return DMUON_ERR_INVALID_ARG; }
  if (count == 0) return DMUON_OK;
  int rc = check_device();
  if (rc) return rc;
  GemmCall& gc = g_gemm_call;
  bool same = gc.op == op && gc.m == m && gc.n == n && gc.variant == variant && gc.in0.size() == static_cast<size_t>(count);
  for (int i = 0; same && i < count; ++i)
    same = gc.in0[i] == in0[i] && gc.out[i] == out[i] && (op != OP_BX || gc.in1[i] == in1[i]);
  if (!same) {
    if (gc.d_probs) cudaFree(gc.d_probs);
    if (gc.d_units) cudaFree(gc.d_units);
    gc = GemmCall();
    std::vector<GemmProblem> probs(count);
    for (int i = 0; i < count; ++i) {
      if (!in0[i] || !out[i] || (op == OP_BX && !in1[i])) { set_error("dmuon_ns_gemm: problem %d has a null pointer", i); return DMUON_ERR_INVALID_ARG; }
      if (op == OP_SYRK) rc = fill_problem(probs[i], OP_SYRK, in0[i], m, n, in0[i], m, n, nullptr, out[i], m);
      else if (op == OP_SQ) rc = fill_problem(probs[i], OP_SQ, in0[i], m, m, in0[i], m, m, in0[i], out[i], m);
      else rc = fill_problem(probs[i], OP_BX, in0[i], m, m, in1[i], m, n, in1[i], out[i], n);
      if (rc) return rc;
    }
    std::vector<TileUnit> units = make_units(static_cast<GemmOp>(op), m / kBlk, n / kBlk, variant_config(variant < 0 ? 0 : variant));
    DMUON_CUDA_CHECK(cudaMalloc(&gc.d_probs, probs.size() * sizeof(GemmProblem)));
    DMUON_CUDA_CHECK(cudaMalloc(&gc.d_units, units.size() * sizeof(TileUnit)));
    DMUON_CUDA_CHECK(cudaMemcpy(gc.d_probs, probs.data(), probs.size() * sizeof(GemmProblem), cudaMemcpyHostToDevice));
    DMUON_CUDA_CHECK(cudaMemcpy(gc.d_units, units.data(), units.size() * sizeof(TileUnit), cudaMemcpyHostToDevice));
    gc.units = static_cast<int>(units.size());
    gc.op = op; gc.m = m; gc.n = n; gc.variant = variant;
    gc.in0.assign(in0, in0 + count);
    gc.out.assign(out, out + count);
    if (op == OP_BX) gc.in1.assign(in1, in1 + count);
  }
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  GemmLaunch L;
  L.op = static_cast<GemmOp>(op);
  L.problems = gc.d_probs;
  L.units = gc.d_units;
  L.units_per_problem = gc.units;
  L.num_problems = count;
  L.k_blocks = (op == OP_SYRK ? n : m) / kBlkK;
  L.m_blocks = m / kBlk;
  L.n_blocks = (op == OP_BX ? n : m) / kBlk;
  L.pair = variant_config(variant < 0 ? 0 : variant).pair;
  L.quad = variant_config(variant < 0 ? 0 : variant).quad;
  L.alpha = alpha;
  L.beta = beta;
  L.beta2 = 0.f;
  L.grid = sms;
  static const char* kNames[3] = {"ns_syrk_xxt", "ns_sq_poly", "ns_bx_update"};
  ProfScope ps(kNames[op], stream);
  return launch_ns_gemm(L, stream);
}

DMUON_API int dmuon_ns_sym_mm(const void* const* a, const void* const* b, const void* const* d, const void* const* d2,
                              void* const* out, int32_t m, int32_t count, float alpha, float beta, float beta2,
                              int32_t variant, dmuon_stream_t stream_) {
  cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
  if (count < 0 || (count > 0 && (!a || !b || !out)) || (d2 && !d)) { set_error("dmuon_ns_sym_mm: null argument"); return DMUON_ERR_INVALID_ARG; }
  if (m <= 0 || m % kBlk) { set_error("dmuon_ns_sym_mm: m must be a positive multiple of 128 (got %d)", m); return DMUON_ERR_INVALID_ARG; }
  if (variant < -1 || (variant >= 0 && !variant_valid(OP_SQ, variant))) { set_error("dmuon_ns_sym_mm: variant %d is not defined", variant); return DMUON_ERR_INVALID_ARG; }
  if (count == 0) return DMUON_OK;
  int rc = check_device();
  if (rc) return rc;
  const GemmOp op = d2 ? OP_SQ2 : d ? OP_SQ : OP_SYRK;
  std::vector<GemmProblem> probs(count);
  for (int i = 0; i < count; ++i) {
    if (!a[i] || !b[i] || !out[i] || (d && !d[i]) || (d2 && !d2[i])) { set_error("dmuon_ns_sym_mm: problem %d has a null pointer", i); return DMUON_ERR_INVALID_ARG; }
    if ((rc = fill_problem(probs[i], op, a[i], m, m, b[i], m, m, d ? d[i] : nullptr, out[i], m, d2 ? d2[i] : nullptr))) return rc;
  }
  const TileConfig cfg = variant_config(variant < 0 ? 0 : variant);
  std::vector<TileUnit> units = make_units(OP_SQ, m / kBlk, m / kBlk, cfg);
  GemmProblem* d_probs = nullptr;
  TileUnit* d_units = nullptr;
  DMUON_CUDA_CHECK(cudaMalloc(&d_probs, probs.size() * sizeof(GemmProblem)));
  DMUON_CUDA_CHECK(cudaMalloc(&d_units, units.size() * sizeof(TileUnit)));
  DMUON_CUDA_CHECK(cudaMemcpy(d_probs, probs.data(), probs.size() * sizeof(GemmProblem), cudaMemcpyHostToDevice));
  DMUON_CUDA_CHECK(cudaMemcpy(d_units, units.data(), units.size() * sizeof(TileUnit), cudaMemcpyHostToDevice));
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  GemmLaunch L;
  L.op = op;
  L.problems = d_probs;
  L.units = d_units;
  L.units_per_problem = static_cast<int>(units.size());
  L.num_problems = count;
  L.k_blocks = m / kBlkK;
  L.m_blocks = m / kBlk;
  L.n_blocks = m / kBlk;
  L.pair = cfg.pair;
  L.quad = cfg.quad;
  L.alpha = alpha;
  L.beta = beta;
  L.beta2 = beta2;
  L.grid = sms;
  {
    ProfScope ps("ns_gram_mm", stream);
    rc = launch_ns_gemm(L, stream);
  }
  cudaError_t e = cudaStreamSynchronize(stream);
  cudaFree(d_probs);
  cudaFree(d_units);
  if (rc) return rc;
  if (e != cudaSuccess) { set_error("dmuon_ns_sym_mm: %s", cudaGetErrorString(e)); return DMUON_ERR_CUDA; }
  return DMUON_OK;
}

DMUON_API void dmuon_shutdown(void) {
  cudaDeviceSynchronize();
  cudaGetLastError();
  fold_profile();
  g_host.release();
  drop_plans();
  g_last_plan = nullptr;
  if (g_gemm_call.d_probs) cudaFree(g_gemm_call.d_probs);
  if (g_gemm_call.d_units) cudaFree(g_gemm_call.d_units);
  g_gemm_call = GemmCall();
  for (cudaEvent_t e : g_event_pool) cudaEventDestroy(e);
  g_event_pool.clear();
  g_prof_acc.clear();
  g_launches = 0;
}

}  // extern "C"
