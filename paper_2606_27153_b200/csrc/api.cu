// C ABI of libdmuon (include/dmuon.h): argument validation, options, error strings, profiling events, and the
// enqueue order of the Muon step, bucket by bucket:
//   momentum+Nesterov+cast+sumsq -> norms -> normalise/cast -> the bucket's NS program (Gram product, polynomial and
//   Gram-space products, X updates; the last X update applies the weight update in its epilogue).
// (Eq. 1, Eq. 2, Alg. 1 l.12-16.)
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>

#include "planner.h"

namespace dmuon {

namespace {

thread_local char g_err[512] = "";
// One lock around every entry point: plans, options, workspaces and caches are process-wide, so calls from several host
// threads are serialised here (recursive: dmuon_muon_step_host and dmuon_measure_cost re-enter the step).
std::recursive_mutex g_mu;
#define DMUON_LOCK std::lock_guard<std::recursive_mutex> dmuon_lock_(g_mu)
Options g_opt;
uint64_t g_last_plan = 0;        // id of the plan of the most recent step / ns call (for dmuon_read_ns_output)
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
long long g_launches = 0;                         // kernels launched (copies are not counted)

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

// Pinned snapshots for asynchronous table uploads.  An upload must carry the values of ITS call (the host mirror is
// patched again by the next call, possibly before the copy has run), so every upload copies the mirror into a pinned
// buffer of its own; the buffer returns to the pool once the stream has passed the copy.  Under stream capture the
// buffer belongs to the graph (the memcpy node re-reads it at every replay) and is never reused.
struct PinnedBuf {
  void* ptr = nullptr;
  size_t bytes = 0;
  cudaEvent_t done = nullptr;
  bool permanent = false;
};
std::vector<PinnedBuf> g_pinned;

int upload_snapshot(void* dst, const void* src, size_t bytes, cudaStream_t stream) {
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  cudaStreamIsCapturing(stream, &cap);
  const bool capturing = cap != cudaStreamCaptureStatusNone;
  PinnedBuf* buf = nullptr;
  if (!capturing) {
    for (PinnedBuf& b : g_pinned)
      if (!b.permanent && b.bytes >= bytes && cudaEventQuery(b.done) == cudaSuccess) { buf = &b; break; }
    cudaGetLastError();      // cudaErrorNotReady from the queries is not an error
  }
  if (!buf) {
    // allocation is not a capturable operation: step out of the capture's error mode for it (the memcpy below is what
    // the graph records)
    cudaStreamCaptureMode mode = cudaStreamCaptureModeRelaxed;
    if (capturing) cudaThreadExchangeStreamCaptureMode(&mode);
    PinnedBuf nb;
    nb.bytes = bytes < 4096 ? 4096 : bytes;
    cudaError_t e1 = cudaMallocHost(&nb.ptr, nb.bytes);
    cudaError_t e2 = e1 == cudaSuccess ? cudaEventCreateWithFlags(&nb.done, cudaEventDisableTiming) : e1;
    if (capturing) cudaThreadExchangeStreamCaptureMode(&mode);
    if (e1 != cudaSuccess) { cudaGetLastError(); set_error("pinned allocation of %zu bytes failed", nb.bytes); return DMUON_ERR_OOM; }
    if (e2 != cudaSuccess) { cudaFreeHost(nb.ptr); cudaGetLastError(); set_error("event creation failed"); return DMUON_ERR_CUDA; }
    g_pinned.push_back(nb);
    buf = &g_pinned.back();
  }
  memcpy(buf->ptr, src, bytes);
  DMUON_CUDA_CHECK(cudaMemcpyAsync(dst, buf->ptr, bytes, cudaMemcpyHostToDevice, stream));
  if (!capturing) DMUON_CUDA_CHECK(cudaEventRecord(buf->done, stream));
  else buf->permanent = true;
  return DMUON_OK;
}

void release_pinned() {
  for (PinnedBuf& b : g_pinned) {
    if (b.done) cudaEventDestroy(b.done);
    if (b.ptr) cudaFreeHost(b.ptr);
  }
  g_pinned.clear();
}

// Patch the per-call pointers into the plan's records (host mirror) and upload them if anything changed.
int bind_pointers(Plan& plan, void* const* w, const void* const* g, void* const* m, int steps, const float* coeffs,
                  bool per_step, cudaStream_t stream, void* const* masters = nullptr) {
  const int count = static_cast<int>(plan.mats.size());
  bool dirty = false;
  std::vector<int> parity(plan.shapes_tbl.size());
  for (size_t s = 0; s < plan.shapes_tbl.size(); ++s)
    parity[s] = result_parity(plan, plan.shapes_tbl[s], steps, coeffs, per_step, g_opt);
  for (int i = 0; i < count; ++i) {
    const MatrixInfo& info = plan.mats[i];
    MatRec& r = plan.h_recs[info.rec];
    void* gi = g ? const_cast<void*>(g[i]) : nullptr;
    void* mi = m ? m[i] : nullptr;
    float* w32 = masters ? static_cast<float*>(masters[i]) : nullptr;
    if (r.W != w[i] || r.G != gi || r.M != mi || r.W32 != w32) dirty = true;
    r.W32 = w32;
    r.W = w[i];
    r.G = gi;
    r.M = mi;
    const int sh = plan.buckets[info.bucket].shape;
    const void* o = parity[sh] ? r.U : r.X0;       // X0 in Q (= rec.X0); each block swaps buffers; P = rec.U
    if (r.O != o) dirty = true;
    r.O = o;
  }
  // A graph replay rewrites d_recs from its own pinned snapshot WITHOUT touching the host mirror, so once a capture
  // has recorded a call on this plan the mirror no longer says what the device holds: from then on every call uploads.
  // A capture always records its upload, so that a replay never runs on what another call left in d_recs.
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  cudaStreamIsCapturing(stream, &cap);
  if (cap != cudaStreamCaptureStatusNone) plan.captured = true;
  if ((dirty || plan.captured) && count > 0)
    return upload_snapshot(plan.d_recs, plan.h_recs.data(), sizeof(MatRec) * count, stream);
  return DMUON_OK;
}

// coefficients of the Muon-step entry points: option "coeffs_sched" (one triple per step) or "coeffs" at every step
const float* step_coeffs(bool* per_step) {
  if (!g_opt.sched.empty() && static_cast<int>(g_opt.sched.size()) == 3 * g_opt.steps) {
    *per_step = true;
    return g_opt.sched.data();
  }
  *per_step = false;
  return g_opt.coeffs;
}

int muon_step_device(void* const* params, const void* const* grads, void* const* momenta, const int32_t* shapes,
                     int32_t count, float lr, float mu, float wd, cudaStream_t stream, Plan** plan_out,
                     void* const* masters = nullptr) {
  if (!g_opt.sched.empty() && static_cast<int>(g_opt.sched.size()) != 3 * g_opt.steps) {
    set_error("option coeffs_sched holds %zu triples but steps = %d", g_opt.sched.size() / 3, g_opt.steps);
    return DMUON_ERR_INVALID_ARG;
  }
  Plan* plan = nullptr;
  int rc = get_plan(shapes, count, g_opt, g_ext_ws, g_ext_ws_bytes, stream, &plan);
  if (rc) return rc;
  if (plan_out) *plan_out = plan;
  g_last_plan = plan->id;
  bool per_step = false;
  const float* coeffs = step_coeffs(&per_step);
  if ((rc = bind_pointers(*plan, params, grads, momenta, g_opt.steps, coeffs, per_step, stream, masters))) return rc;
  const bool master = masters != nullptr;
  FinalEpilogue fin;
  fin.epi = master ? EPI_APPLY_MASTER : EPI_APPLY;
  fin.lr = lr;
  fin.lrwd = lr * wd;
  fin.store_c = plan->keep_o;
  plan->o_valid = plan->keep_o || (plan->buckets.size() == 1 && !bucket_fuses(*plan, plan->shapes_tbl[plan->buckets[0].shape], g_opt.steps, g_opt));
  for (size_t b = 0; b < plan->buckets.size(); ++b) {
    const BucketPlan& bp = plan->buckets[b];
    const ElemTables& T = bp.tables;
    if ((rc = launch_momentum(T, mu, /*exact=*/plan->fp32, stream))) return rc;
    if ((rc = launch_finalize_norms(T, g_opt.eps, stream))) return rc;
    if ((rc = launch_normalize(T, /*from_user=*/false, plan->fp32, stream))) return rc;
    if ((rc = run_ns_bucket(*plan, static_cast<int>(b), g_opt.steps, coeffs, per_step, g_opt, fin, stream))) return rc;
    if (!bucket_fuses(*plan, plan->shapes_tbl[bp.shape], g_opt.steps, g_opt))
      if ((rc = launch_apply(T, lr, wd, plan->fp32, master, stream))) return rc;
  }
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
  g_last_plan = plan->id;
  if ((rc = bind_pointers(*plan, ptrs, nullptr, nullptr, steps, coeffs, per_step, stream))) return rc;
  FinalEpilogue fin;
  fin.epi = EPI_BF16;
  fin.store_c = plan->keep_o;
  plan->o_valid = plan->keep_o || (plan->buckets.size() == 1 && !bucket_fuses(*plan, plan->shapes_tbl[plan->buckets[0].shape], steps, g_opt));
  for (size_t b = 0; b < plan->buckets.size(); ++b) {
    const BucketPlan& bp = plan->buckets[b];
    const ElemTables& T = bp.tables;
    if ((rc = launch_sumsq(T, stream))) return rc;
    if ((rc = launch_finalize_norms(T, g_opt.eps, stream))) return rc;
    if ((rc = launch_normalize(T, /*from_user=*/true, plan->fp32, stream))) return rc;
    if ((rc = run_ns_bucket(*plan, static_cast<int>(b), steps, coeffs, per_step, g_opt, fin, stream))) return rc;
    if (!bucket_fuses(*plan, plan->shapes_tbl[bp.shape], steps, g_opt))
      if ((rc = launch_store_ns(T, plan->fp32, stream))) return rc;
  }
  return DMUON_OK;
}

// ---- state of dmuon_muon_step_host: a ring of three device staging slots (W | G | M of one group of matrices each),
//      copy streams, events (one shape set at a time)
struct HostCtx {
  std::vector<int32_t> shapes;
  int device = -1;
  uint8_t* stage = nullptr;
  std::vector<size_t> off;      // per matrix offset of W inside its group's slot; G at + third, M at + 2 * third
  size_t third = 0;             // bytes of one of W / G / M of a group
  int group = 0;                // matrices per group
  int slots = 0;                // staging slots
  int opt_groups = 0, opt_slots = 0;   // the option values this context was built for
  cudaStream_t s_in = nullptr, s_out = nullptr;
  std::vector<cudaEvent_t> ev;  // [3 g] copy-in done, [3 g + 1] step done, [3 g + 2] copy-out done, then start / end
  int release() {
    if (stage || s_in) cudaDeviceSynchronize();
    if (stage) cudaFree(stage);
    if (s_in) cudaStreamDestroy(s_in);
    if (s_out) cudaStreamDestroy(s_out);
    for (cudaEvent_t e : ev) if (e) cudaEventDestroy(e);
    cudaGetLastError();
    *this = HostCtx();
    return DMUON_OK;
  }
} g_host;

// ---- dmuon_ns_gemm table cache (one entry: the last argument set)
struct GemmCall {
  std::vector<const void*> in0, in1;
  std::vector<void*> out;
  int op = -1, m = 0, n = 0, variant = -2, device = -1;
  GemmProblem* d_probs = nullptr;
  TileUnit* d_units = nullptr;
  int units = 0;
} g_gemm_call;

// ---- dmuon_adamw_step table cache (one entry: the last tensor list)
struct AdamCall {
  std::vector<AdamRec> recs;
  int device = -1;
  AdamRec* d_recs = nullptr;
  int64_t* d_prefix = nullptr;
  int64_t chunks = 0;
  void release() {
    if (d_recs) cudaFree(d_recs);
    if (d_prefix) cudaFree(d_prefix);
    *this = AdamCall();
  }
} g_adam_call;

int current_sms() {
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  return sms;
}

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

DMUON_API const char* dmuon_version(void) { return "libdmuon 0.2 (sm_100a)"; }

DMUON_API const char* dmuon_last_error(void) { return g_err; }

DMUON_API int dmuon_set_option(const char* key, const char* value) {
  DMUON_LOCK;
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
  if (k == "coeffs_sched") {
    // "a0,b0,c0;a1,b1,c1;..." -- one triple per NS step of the Muon-step entry points; "" = off
    std::vector<float> sched;
    const char* p = value;
    while (*p) {
      float a, b, c;
      int used = 0;
      if (sscanf(p, " %f , %f , %f %n", &a, &b, &c, &used) != 3) { set_error("option coeffs_sched: expected 'a,b,c;a,b,c;...', got '%s'", value); return DMUON_ERR_INVALID_ARG; }
      sched.push_back(a); sched.push_back(b); sched.push_back(c);
      p += used;
      if (*p == ';') ++p;
      else if (*p) { set_error("option coeffs_sched: unexpected '%c' in '%s'", *p, value); return DMUON_ERR_INVALID_ARG; }
    }
    if (sched.size() / 3 > 64) { set_error("option coeffs_sched: more than 64 steps"); return DMUON_ERR_INVALID_ARG; }
    g_opt.sched = sched;
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
  if (k == "fuse_epilogue") { if (as_bool(&g_opt.fuse)) return DMUON_OK; set_error("option fuse_epilogue: bad value '%s'", value); return DMUON_ERR_INVALID_ARG; }
  if (k == "small_fused") { if (as_bool(&g_opt.small_fused)) return DMUON_OK; set_error("option small_fused: bad value '%s'", value); return DMUON_ERR_INVALID_ARG; }
  if (k == "graphs_destroyed") {
    // the caller states that every CUDA graph captured from this library's calls has been destroyed: plans and the
    // workspace may be evicted / moved again, and eager calls stop re-uploading their tables
    bool yes = false;
    if (!as_bool(&yes) || !yes) { set_error("option graphs_destroyed: the only value is 1"); return DMUON_ERR_INVALID_ARG; }
    forget_captures();
    for (PinnedBuf& b : g_pinned) b.permanent = false;      // the graphs' upload snapshots can be reused
    return DMUON_OK;
  }
  if (k == "keep_ns_output") { if (as_bool(&g_opt.keep_o)) return DMUON_OK; set_error("option keep_ns_output: bad value '%s'", value); return DMUON_ERR_INVALID_ARG; }
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
  if (k == "chunk_mb") {
    char* end = nullptr;
    long long mb = strtoll(value, &end, 10);
    if (end == value || *end || mb < 1) { set_error("option chunk_mb: bad value '%s'", value); return DMUON_ERR_INVALID_ARG; }
    g_opt.chunk_bytes = static_cast<size_t>(mb) << 20;
    return DMUON_OK;
  }
  if (k == "program") {
    if (v == "0" || v == "1" || v == "auto") { g_opt.program = v == "auto" ? 2 : (v == "1" ? 1 : 0); return DMUON_OK; }
    set_error("option program: expected '0', '1' or 'auto', got '%s'", value);
    return DMUON_ERR_INVALID_ARG;
  }
  if (k == "l2_group_mb") {
    char* end = nullptr;
    long long mb = strtoll(value, &end, 10);
    if (end == value || *end || mb < 1 || mb > (1 << 20)) { set_error("option l2_group_mb: bad value '%s'", value); return DMUON_ERR_INVALID_ARG; }
    g_opt.l2_group_bytes = static_cast<size_t>(mb) << 20;
    return DMUON_OK;
  }
  if (k == "tune_ms") {
    char* end = nullptr;
    float ms = strtof(value, &end);
    if (end == value || *end || !(ms >= 0.f) || ms > 10000.f) { set_error("option tune_ms: bad value '%s'", value); return DMUON_ERR_INVALID_ARG; }
    g_opt.tune_ms = ms;
    return DMUON_OK;
  }
  if (k == "host_pipeline") {
    int a, b;
    char tail;
    if (sscanf(value, " %d , %d %c", &a, &b, &tail) != 2 || a < 1 || b < 1 || a > 64 || b > 64) { set_error("option host_pipeline: expected 'groups,slots' in 1..64, got '%s'", value); return DMUON_ERR_INVALID_ARG; }
    g_opt.host_groups = a;
    g_opt.host_slots = b;
    return DMUON_OK;
  }
  if (k == "cache_path") { g_opt.cache_path = v; g_opt.cache_path_set = true; return DMUON_OK; }
  set_error("dmuon_set_option: unknown key '%s'", key);
  return DMUON_ERR_INVALID_ARG;
}

DMUON_API int dmuon_ns_batched(void* const* ptrs, const int32_t* shapes, int32_t count, int32_t steps,
                               const float* coeffs, dmuon_stream_t stream) {
  DMUON_LOCK;
  return ns_batched_impl(ptrs, shapes, count, steps, coeffs, false, reinterpret_cast<cudaStream_t>(stream));
}

DMUON_API int dmuon_ns_batched_sched(void* const* ptrs, const int32_t* shapes, int32_t count, int32_t steps,
                                     const float* coeffs, dmuon_stream_t stream) {
  DMUON_LOCK;
  return ns_batched_impl(ptrs, shapes, count, steps, coeffs, true, reinterpret_cast<cudaStream_t>(stream));
}

DMUON_API int dmuon_muon_step(void* const* params, const void* const* grads, void* const* momenta,
                              const int32_t* shapes, int32_t count, float lr, float mu, float wd,
                              dmuon_stream_t stream) {
  DMUON_LOCK;
  int rc = validate(reinterpret_cast<const void* const*>(params), grads, reinterpret_cast<const void* const*>(momenta),
                    shapes, count, "dmuon_muon_step");
  if (rc || count == 0) return rc;
  if (!grads || !momenta) { set_error("dmuon_muon_step: null argument"); return DMUON_ERR_INVALID_ARG; }
  return muon_step_device(params, grads, momenta, shapes, count, lr, mu, wd, reinterpret_cast<cudaStream_t>(stream), nullptr);
}

DMUON_API int dmuon_muon_step_master(void* const* params, void* const* masters, const void* const* grads,
                                     void* const* momenta, const int32_t* shapes, int32_t count, float lr, float mu,
                                     float wd, dmuon_stream_t stream) {
  DMUON_LOCK;
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
// so that every group has the same shape list and shares one plan and one workspace.  Three device staging slots
// rotate: group g's host->device copies (copy-in stream), the step of group g-1 (caller's stream) and the device->host
// copies of group g-2 (copy-out stream) overlap; PCIe carries both directions at once.
DMUON_API int dmuon_muon_step_host(void* const* params_host, const void* const* grads_host, void* const* momenta_host,
                                   const int32_t* shapes, int32_t count, float lr, float mu, float wd,
                                   dmuon_stream_t stream_) {
  DMUON_LOCK;
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
  int dev = 0;
  cudaGetDevice(&dev);
  HostCtx& hc = g_host;
  if (hc.device != dev || hc.opt_groups != g_opt.host_groups || hc.opt_slots != g_opt.host_slots ||
      hc.shapes.size() != static_cast<size_t>(2 * count) ||
      memcmp(hc.shapes.data(), shapes, sizeof(int32_t) * 2 * count) != 0) {
    if ((rc = hc.release())) return rc;
    HostCtx nc;                                        // committed to g_host only when fully set up
    // smallest period of the shape pattern, then the smallest number of periods per group that gives <= host_groups groups
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
      if (periods % d == 0 && periods / d <= g_opt.host_groups) { per_group = d; break; }
    nc.group = per_group * period;
    size_t off = 0;
    nc.off.resize(nc.group);
    for (int i = 0; i < nc.group; ++i) {
      nc.off[i] = off;
      off += (static_cast<size_t>(shapes[2 * i]) * shapes[2 * i + 1] * 2 + 255) / 256 * 256;
    }
    nc.third = off;
    const int groups = count / nc.group;
    const int slots = groups < g_opt.host_slots ? groups : g_opt.host_slots;
    nc.slots = slots;
    nc.opt_groups = g_opt.host_groups;
    nc.opt_slots = g_opt.host_slots;
    void* p = nullptr;
    cudaError_t e = cudaMalloc(&p, 3 * off * slots);
    if (e != cudaSuccess) { cudaGetLastError(); set_error("staging allocation of %zu bytes failed", 3 * off * slots); return DMUON_ERR_OOM; }
    nc.stage = static_cast<uint8_t*>(p);
    nc.ev.assign(3 * groups + 2, nullptr);
    bool ok = cudaStreamCreateWithFlags(&nc.s_in, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&nc.s_out, cudaStreamNonBlocking) == cudaSuccess;
    for (cudaEvent_t& ev : nc.ev) ok = ok && cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) == cudaSuccess;
    if (!ok) { nc.release(); set_error("dmuon_muon_step_host: stream / event creation failed"); return DMUON_ERR_CUDA; }
    nc.device = dev;
    nc.shapes.assign(shapes, shapes + 2 * count);
    hc = nc;
  }
  const int groups = count / hc.group;
  const int gsz = hc.group;
  cudaEvent_t ev_start = hc.ev[3 * groups], ev_end = hc.ev[3 * groups + 1];
  std::vector<void*> w(gsz), m(gsz);
  std::vector<const void*> g(gsz);
  auto bytes_of = [&](int i) { return static_cast<size_t>(shapes[2 * i]) * shapes[2 * i + 1] * 2; };
  bool enqueued = false;
  // every exit after the first enqueue waits for what was queued: the caller's host buffers must not be written later
  auto fail = [&](int code) {
    if (enqueued) { cudaDeviceSynchronize(); cudaGetLastError(); }
    hc.release();
    return code;
  };
#define DMUON_HOST_CHECK(expr)                                                                                  \
  do {                                                                                                          \
    cudaError_t _e = (expr);                                                                                    \
    if (_e != cudaSuccess) { set_error("%s failed: %s", #expr, cudaGetErrorString(_e)); return fail(DMUON_ERR_CUDA); } \
  } while (0)
  DMUON_HOST_CHECK(cudaEventRecord(ev_start, stream));            // copies start after the caller's earlier work
  DMUON_HOST_CHECK(cudaStreamWaitEvent(hc.s_in, ev_start, 0));
  for (int gi = 0; gi < groups; ++gi) {
    const int b = gi * gsz;
    uint8_t* slot = hc.stage + static_cast<size_t>(gi % hc.slots) * 3 * hc.third;
    for (int i = 0; i < gsz; ++i) {
      w[i] = slot + hc.off[i];
      g[i] = slot + hc.third + hc.off[i];
      m[i] = slot + 2 * hc.third + hc.off[i];
    }
    if (gi >= hc.slots) DMUON_HOST_CHECK(cudaStreamWaitEvent(hc.s_in, hc.ev[3 * (gi - hc.slots) + 2], 0));   // slot drained
    for (int i = 0; i < gsz; ++i) {
      DMUON_HOST_CHECK(cudaMemcpyAsync(w[i], params_host[b + i], bytes_of(b + i), cudaMemcpyHostToDevice, hc.s_in));
      enqueued = true;
      DMUON_HOST_CHECK(cudaMemcpyAsync(const_cast<void*>(g[i]), grads_host[b + i], bytes_of(b + i), cudaMemcpyHostToDevice, hc.s_in));
      DMUON_HOST_CHECK(cudaMemcpyAsync(m[i], momenta_host[b + i], bytes_of(b + i), cudaMemcpyHostToDevice, hc.s_in));
    }
    DMUON_HOST_CHECK(cudaEventRecord(hc.ev[3 * gi], hc.s_in));
    DMUON_HOST_CHECK(cudaStreamWaitEvent(stream, hc.ev[3 * gi], 0));
    if ((rc = muon_step_device(w.data(), g.data(), m.data(), shapes + 2 * b, gsz, lr, mu, wd, stream, nullptr))) return fail(rc);
    DMUON_HOST_CHECK(cudaEventRecord(hc.ev[3 * gi + 1], stream));
    DMUON_HOST_CHECK(cudaStreamWaitEvent(hc.s_out, hc.ev[3 * gi + 1], 0));
    for (int i = 0; i < gsz; ++i) {
      DMUON_HOST_CHECK(cudaMemcpyAsync(params_host[b + i], w[i], bytes_of(b + i), cudaMemcpyDeviceToHost, hc.s_out));
      DMUON_HOST_CHECK(cudaMemcpyAsync(momenta_host[b + i], m[i], bytes_of(b + i), cudaMemcpyDeviceToHost, hc.s_out));
    }
    DMUON_HOST_CHECK(cudaEventRecord(hc.ev[3 * gi + 2], hc.s_out));
  }
  DMUON_HOST_CHECK(cudaEventRecord(ev_end, hc.s_out));
  DMUON_HOST_CHECK(cudaStreamWaitEvent(stream, ev_end, 0));      // the caller's stream sees the results
#undef DMUON_HOST_CHECK
  return DMUON_OK;
}

// Non-matrix parameters (Alg. 1 l.16): decoupled AdamW, one flat launch over all tensors.
DMUON_API int dmuon_adamw_step(void* const* params, const void* const* grads, void* const* exp_avg,
                               void* const* exp_avg_sq, const int64_t* numel, int32_t count, float lr, float beta1,
                               float beta2, float eps, float wd, int32_t step, dmuon_stream_t stream_) {
  DMUON_LOCK;
  cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
  if (count < 0) { set_error("dmuon_adamw_step: count < 0"); return DMUON_ERR_INVALID_ARG; }
  if (count == 0) return DMUON_OK;
  if (!params || !grads || !exp_avg || !exp_avg_sq || !numel) { set_error("dmuon_adamw_step: null argument"); return DMUON_ERR_INVALID_ARG; }
  if (step < 1) { set_error("dmuon_adamw_step: step counts from 1 (got %d)", step); return DMUON_ERR_INVALID_ARG; }
  if (!(beta1 >= 0.f && beta1 < 1.f) || !(beta2 >= 0.f && beta2 < 1.f) || !(eps >= 0.f)) { set_error("dmuon_adamw_step: beta1, beta2 must be in [0, 1), eps >= 0"); return DMUON_ERR_INVALID_ARG; }
  for (int i = 0; i < count; ++i) {
    if (numel[i] <= 0) { set_error("dmuon_adamw_step: tensor %d has %lld elements", i, static_cast<long long>(numel[i])); return DMUON_ERR_INVALID_ARG; }
    const void* ptrs[4] = {params[i], grads[i], exp_avg[i], exp_avg_sq[i]};
    for (const void* p : ptrs) {
      if (!p) { set_error("dmuon_adamw_step: tensor %d has a null pointer", i); return DMUON_ERR_INVALID_ARG; }
      if (reinterpret_cast<uintptr_t>(p) & 15) { set_error("dmuon_adamw_step: tensor %d pointer %p is not 16-byte aligned", i, p); return DMUON_ERR_INVALID_ARG; }
    }
  }
  int rc = check_device();
  if (rc) return rc;
  int dev = 0;
  cudaGetDevice(&dev);
  AdamCall& ac = g_adam_call;
  bool same = ac.device == dev && ac.recs.size() == static_cast<size_t>(count);
  for (int i = 0; same && i < count; ++i)
    same = ac.recs[i].p == params[i] && ac.recs[i].g == grads[i] && ac.recs[i].m == exp_avg[i] &&
           ac.recs[i].v == exp_avg_sq[i] && ac.recs[i].numel == numel[i];
  if (!same) {
    ac.release();
    std::vector<AdamRec> recs(count);
    std::vector<int64_t> prefix(count + 1, 0);
    for (int i = 0; i < count; ++i) {
      recs[i] = AdamRec{params[i], grads[i], static_cast<float*>(exp_avg[i]), static_cast<float*>(exp_avg_sq[i]), numel[i]};
      prefix[i + 1] = prefix[i] + (numel[i] + kFlatChunk - 1) / kFlatChunk;
    }
    DMUON_CUDA_CHECK(cudaMalloc(&ac.d_recs, recs.size() * sizeof(AdamRec)));
    DMUON_CUDA_CHECK(cudaMalloc(&ac.d_prefix, prefix.size() * sizeof(int64_t)));
    DMUON_CUDA_CHECK(cudaMemcpy(ac.d_recs, recs.data(), recs.size() * sizeof(AdamRec), cudaMemcpyHostToDevice));
    DMUON_CUDA_CHECK(cudaMemcpy(ac.d_prefix, prefix.data(), prefix.size() * sizeof(int64_t), cudaMemcpyHostToDevice));
    ac.recs = recs;
    ac.chunks = prefix[count];
    ac.device = dev;
  }
  AdamScalars sc;
  sc.lr = lr; sc.beta1 = beta1; sc.beta2 = beta2; sc.eps = eps; sc.wd = wd;
  sc.inv_bc1 = static_cast<float>(1.0 / (1.0 - std::pow(static_cast<double>(beta1), step)));
  sc.inv_sqrt_bc2 = static_cast<float>(1.0 / std::sqrt(1.0 - std::pow(static_cast<double>(beta2), step)));
  return launch_adamw(ac.d_recs, ac.d_prefix, count, ac.chunks, sc, stream);
}

// dmuon_adamw_step for callers that must not touch the CUDA allocator: same kernel, same arithmetic, the work table
// in the library's static device array (elementwise.cu: launch_adamw_static).  No cudaMalloc / cudaFree / cudaMallocHost
// and no event creation on this path (the profile option does not record it).
DMUON_API int dmuon_adamw_step_noalloc(void* const* params, const void* const* grads, void* const* exp_avg,
                                       void* const* exp_avg_sq, const int64_t* numel, int32_t count, float lr,
                                       float beta1, float beta2, float eps, float wd, int32_t step,
                                       dmuon_stream_t stream_) {
  DMUON_LOCK;
  static const char* const fn = "dmuon_adamw_step_noalloc";
  if (count < 0) { set_error("%s: count < 0", fn); return DMUON_ERR_INVALID_ARG; }
  if (count == 0) return DMUON_OK;
  if (count > DMUON_ADAMW_NOALLOC_MAX_TENSORS) {
    set_error("%s: %d tensors in one call, the built-in table holds DMUON_ADAMW_NOALLOC_MAX_TENSORS = %d (split the list, or use dmuon_adamw_step)",
              fn, count, DMUON_ADAMW_NOALLOC_MAX_TENSORS);
    return DMUON_ERR_INVALID_ARG;
  }
  if (!params || !grads || !exp_avg || !exp_avg_sq || !numel) { set_error("%s: null argument", fn); return DMUON_ERR_INVALID_ARG; }
  if (step < 1) { set_error("%s: step counts from 1 (got %d)", fn, step); return DMUON_ERR_INVALID_ARG; }
  if (!(beta1 >= 0.f && beta1 < 1.f) || !(beta2 >= 0.f && beta2 < 1.f) || !(eps >= 0.f)) { set_error("%s: beta1, beta2 must be in [0, 1), eps >= 0", fn); return DMUON_ERR_INVALID_ARG; }
  for (int i = 0; i < count; ++i) {
    if (numel[i] <= 0) { set_error("%s: tensor %d has %lld elements", fn, i, static_cast<long long>(numel[i])); return DMUON_ERR_INVALID_ARG; }
    const void* ptrs[4] = {params[i], grads[i], exp_avg[i], exp_avg_sq[i]};
    for (const void* p : ptrs) {
      if (!p) { set_error("%s: tensor %d has a null pointer", fn, i); return DMUON_ERR_INVALID_ARG; }
      if (reinterpret_cast<uintptr_t>(p) & 15) { set_error("%s: tensor %d pointer %p is not 16-byte aligned", fn, i, p); return DMUON_ERR_INVALID_ARG; }
    }
  }
  int rc = check_device();
  if (rc) return rc;
  AdamScalars sc;
  sc.lr = lr; sc.beta1 = beta1; sc.beta2 = beta2; sc.eps = eps; sc.wd = wd;
  sc.inv_bc1 = static_cast<float>(1.0 / (1.0 - std::pow(static_cast<double>(beta1), step)));
  sc.inv_sqrt_bc2 = static_cast<float>(1.0 / std::sqrt(1.0 - std::pow(static_cast<double>(beta2), step)));
  return launch_adamw_static(params, grads, exp_avg, exp_avg_sq, numel, count, sc, reinterpret_cast<cudaStream_t>(stream_));
}

DMUON_API int dmuon_warmup(const int32_t* shapes, int32_t count, dmuon_stream_t stream) {
  DMUON_LOCK;
  if (count < 0 || (count > 0 && !shapes)) { set_error("dmuon_warmup: bad arguments"); return DMUON_ERR_INVALID_ARG; }
  for (int i = 0; i < count; ++i)
    if (shapes[2 * i] <= 0 || shapes[2 * i + 1] <= 0) { set_error("dmuon_warmup: bad shape of matrix %d", i); return DMUON_ERR_INVALID_ARG; }
  if (count == 0) return DMUON_OK;
  Plan* plan = nullptr;
  return get_plan(shapes, count, g_opt, g_ext_ws, g_ext_ws_bytes, reinterpret_cast<cudaStream_t>(stream), &plan);
}

DMUON_API int dmuon_block_schedule(int32_t rows, int32_t cols, int32_t steps, const float* coeffs, int32_t per_step,
                                   int32_t* out, int32_t cap) {
  DMUON_LOCK;
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
  DMUON_LOCK;
  if (count < 0 || steps < 0 || (count > 0 && !shapes)) { set_error("dmuon_describe_plan: bad arguments"); return DMUON_ERR_INVALID_ARG; }
  for (int i = 0; i < count; ++i)
    if (shapes[2 * i] <= 0 || shapes[2 * i + 1] <= 0) { set_error("dmuon_describe_plan: bad shape of matrix %d", i); return DMUON_ERR_INVALID_ARG; }
  std::string s = "{\"buckets\": [";
  char item[256];
  if (count > 0) {
    Plan* plan = nullptr;
    int rc = get_plan(shapes, count, g_opt, g_ext_ws, g_ext_ws_bytes, reinterpret_cast<cudaStream_t>(stream), &plan);
    if (rc) return rc;
    bool per_step = false;
    const float* coeffs = step_coeffs(&per_step);
    if (per_step && steps != g_opt.steps) { per_step = false; coeffs = g_opt.coeffs; }
    bool first = true;
    static const char* kKind[3] = {"wide", "tall", "generic"};
    for (const BucketPlan& bp : plan->buckets) {
      const ShapeTables& st = plan->shapes_tbl[bp.shape];
      const Partition part = plan->fp32 ? Partition(steps, 1)
                                        : choose_partition(steps, coeffs, per_step, st.gram && g_opt.gram_blocks);
      snprintf(item, sizeof item, "%s{\"m\": %d, \"n\": %d, \"kind\": \"%s\", \"count\": %d, \"blocks\": [", first ? "" : ", ",
               st.m_pad, st.n_pad, kKind[st.kind], static_cast<int>(bp.mats.size()));
      s += item;
      for (size_t k = 0; k < part.size(); ++k) s += (k ? ", " : "") + std::to_string(part[k]);
      snprintf(item, sizeof item, "], \"variants\": [%d, %d, %d], \"fused\": %s, \"onchip\": %s, \"program\": %s, \"xscale\": %g, \"gscale\": %g}", st.variant[0],
               st.variant[1], st.variant[2], bucket_fuses(*plan, st, steps, g_opt) ? "true" : "false",
               bucket_onchip(*plan, st, steps, g_opt) ? "true" : "false",
               !bucket_onchip(*plan, st, steps, g_opt) && bucket_program(*plan, st, program_launches(part), g_opt) ? "true" : "false",
               st.xscale, st.gscale);
      s += item;
      first = false;
    }
    snprintf(item, sizeof item, "], \"workspace_bytes\": %zu, \"tune_seconds\": %.4f, \"tune_cache_entries\": %d}", plan->ws_bytes,
             plan->tune_seconds, tune_cache_entries());
    s += item;
  } else {
    s += "], \"workspace_bytes\": 0, \"tune_seconds\": 0, \"tune_cache_entries\": 0}";
  }
  if (buf && len > 0) {
    const size_t n = s.size() < len - 1 ? s.size() : len - 1;
    memcpy(buf, s.data(), n);
    buf[n] = 0;
  }
  return static_cast<int>(s.size());
}

DMUON_API size_t dmuon_workspace_bytes(const int32_t* shapes, int32_t count) {
  DMUON_LOCK;
  if (count <= 0 || !shapes) return 0;
  for (int i = 0; i < count; ++i)
    if (shapes[2 * i] <= 0 || shapes[2 * i + 1] <= 0) return 0;
  return plan_workspace_bytes(shapes, count, g_opt);
}

DMUON_API int dmuon_set_workspace(void* dev_ptr, size_t bytes) {
  DMUON_LOCK;
  if ((dev_ptr == nullptr) != (bytes == 0)) { set_error("dmuon_set_workspace: pointer and size must both be set or both be zero"); return DMUON_ERR_INVALID_ARG; }
  if (reinterpret_cast<uintptr_t>(dev_ptr) & 255) { set_error("dmuon_set_workspace: pointer must be 256-byte aligned"); return DMUON_ERR_INVALID_ARG; }
  if (captured_plans() > 0) {
    set_error("dmuon_set_workspace: a captured CUDA graph refers to the current plans and workspace; destroy the graphs "
              "and set option graphs_destroyed=1 first");
    return DMUON_ERR_INVALID_ARG;
  }
  cudaDeviceSynchronize();
  cudaGetLastError();
  drop_plans();
  g_last_plan = 0;
  g_ext_ws = dev_ptr;
  g_ext_ws_bytes = bytes;
  return DMUON_OK;
}

DMUON_API int dmuon_read_ns_output(int32_t index, float* out_dev, dmuon_stream_t stream) {
  DMUON_LOCK;
  Plan* lp = g_last_plan ? find_plan(g_last_plan) : nullptr;
  if (!lp) { set_error("dmuon_read_ns_output: no step has run (or its plan has been dropped since)"); return DMUON_ERR_INVALID_ARG; }
  Plan& p = *lp;
  if (index < 0 || index >= static_cast<int>(p.mats.size()) || !out_dev) { set_error("dmuon_read_ns_output: bad index or null output"); return DMUON_ERR_INVALID_ARG; }
  if (!p.o_valid) {
    set_error("dmuon_read_ns_output: the last call did not keep the NS results (buckets share one workspace region, fused "
              "epilogues do not store O); set option keep_ns_output=1 before the call");
    return DMUON_ERR_INVALID_ARG;
  }
  const MatrixInfo& mi = p.mats[index];
  const MatRec& r = p.h_recs[mi.rec];
  return launch_export(r.O, out_dev, mi.rows, mi.cols, mi.buf_cols, mi.transposed, p.fp32, r.inv_xscale,
                       reinterpret_cast<cudaStream_t>(stream));
}

DMUON_API int dmuon_profile_reset(void) {
  DMUON_LOCK;
  int rc = fold_profile();
  g_prof_acc.clear();
  g_launches = 0;
  return rc;
}

DMUON_API int dmuon_profile_read(char* buf, size_t len) {
  DMUON_LOCK;
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

DMUON_API int dmuon_ns_gemm_variants(int32_t op) {
  DMUON_LOCK; return (op >= 0 && op < kNumOps && op != OP_SQ2) ? kNumVariants : 0; }

// op: 0 SYRK (in0 = X [m x n]), 1 SQ (in0 = A [m x m]), 2 BX (in0 = B [m x m], in1 = X [m x n]),
//     4 SYRK_T (in0 = Y [n x m]), 5 XB (in0 = B [m x m], in1 = Y [n x m]).
DMUON_API int dmuon_ns_gemm(int32_t op, const void* const* in0, const void* const* in1, void* const* out, int32_t m,
                            int32_t n, int32_t count, float alpha, float beta, int32_t variant, dmuon_stream_t stream_) {
  DMUON_LOCK;
  cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
  if (op < 0 || op >= kNumOps || op == OP_SQ2) { set_error("dmuon_ns_gemm: bad op %d", op); return DMUON_ERR_INVALID_ARG; }
  const bool two = op == OP_BX || op == OP_XB;
  if (count < 0 || (count > 0 && (!in0 || !out || (two && !in1)))) { set_error("dmuon_ns_gemm: null argument"); return DMUON_ERR_INVALID_ARG; }
  if (op == OP_SQ) n = m;
  if (m <= 0 || n <= 0 || m % kBlk || n % kBlk) { set_error("dmuon_ns_gemm: m and n must be positive multiples of 128 (got %d, %d)", m, n); return DMUON_ERR_INVALID_ARG; }
  if (variant < -1 || (variant >= 0 && !variant_valid(static_cast<GemmOp>(op), variant))) { set_error("dmuon_ns_gemm: variant %d is not defined for op %d", variant, op); return DMUON_ERR_INVALID_ARG; }
  if (count == 0) return DMUON_OK;
  int rc = check_device();
  if (rc) return rc;
  int dev = 0;
  cudaGetDevice(&dev);
  const GemmOp gop = static_cast<GemmOp>(op);
  int mb = m / kBlk, nb = m / kBlk;
  if (gop == OP_BX) nb = n / kBlk;
  if (gop == OP_XB) mb = n / kBlk;
  GemmCall& gc = g_gemm_call;
  bool same = gc.device == dev && gc.op == op && gc.m == m && gc.n == n && gc.variant == variant && gc.in0.size() == static_cast<size_t>(count);
  for (int i = 0; same && i < count; ++i)
    same = gc.in0[i] == in0[i] && gc.out[i] == out[i] && (!two || gc.in1[i] == in1[i]);
  if (!same) {
    if (gc.d_probs) cudaFree(gc.d_probs);
    if (gc.d_units) cudaFree(gc.d_units);
    gc = GemmCall();
    std::vector<GemmProblem> probs(count);
    for (int i = 0; i < count; ++i) {
      if (!in0[i] || !out[i] || (two && !in1[i])) { set_error("dmuon_ns_gemm: problem %d has a null pointer", i); return DMUON_ERR_INVALID_ARG; }
      switch (gop) {
        case OP_SYRK: rc = fill_problem(probs[i], OP_SYRK, in0[i], m, n, in0[i], m, n, nullptr, out[i], m); break;
        case OP_SYRK_T: rc = fill_problem(probs[i], OP_SYRK_T, in0[i], n, m, in0[i], n, m, nullptr, out[i], m); break;
        case OP_SQ: rc = fill_problem(probs[i], OP_SQ, in0[i], m, m, in0[i], m, m, in0[i], out[i], m); break;
        case OP_BX: rc = fill_problem(probs[i], OP_BX, in0[i], m, m, in1[i], m, n, in1[i], out[i], n); break;
        default: rc = fill_problem(probs[i], OP_XB, in1[i], n, m, in0[i], m, m, in1[i], out[i], m); break;
      }
      if (rc) return rc;
    }
    std::vector<TileUnit> units = make_units(gop, mb, nb, variant_config(variant < 0 ? 0 : variant));
    DMUON_CUDA_CHECK(cudaMalloc(&gc.d_probs, probs.size() * sizeof(GemmProblem)));
    DMUON_CUDA_CHECK(cudaMalloc(&gc.d_units, units.size() * sizeof(TileUnit)));
    DMUON_CUDA_CHECK(cudaMemcpy(gc.d_probs, probs.data(), probs.size() * sizeof(GemmProblem), cudaMemcpyHostToDevice));
    DMUON_CUDA_CHECK(cudaMemcpy(gc.d_units, units.data(), units.size() * sizeof(TileUnit), cudaMemcpyHostToDevice));
    gc.units = static_cast<int>(units.size());
    gc.op = op; gc.m = m; gc.n = n; gc.variant = variant; gc.device = dev;
    gc.in0.assign(in0, in0 + count);
    gc.out.assign(out, out + count);
    if (two) gc.in1.assign(in1, in1 + count);
  }
  GemmLaunch L;
  L.op = gop;
  L.problems = gc.d_probs;
  L.units = gc.d_units;
  L.units_per_problem = gc.units;
  L.num_problems = count;
  L.k_blocks = ((gop == OP_SYRK || gop == OP_SYRK_T) ? n : m) / kBlkK;
  L.m_blocks = mb;
  L.n_blocks = nb;
  L.pair = variant_config(variant < 0 ? 0 : variant).pair;
  L.epi_warps = variant_config(variant < 0 ? 0 : variant).epi_warps;
  L.alpha = alpha;
  L.beta = beta;
  L.beta2 = 0.f;
  L.grid = current_sms();
  static const char* kNames[kNumOps] = {"ns_syrk_xxt", "ns_sq_poly", "ns_bx_update", "ns_gram_mm", "ns_syrk_xtx", "ns_xb_update"};
  ProfScope ps(kNames[op], stream);
  return launch_ns_gemm(L, stream);
}

DMUON_API int dmuon_ns_sym_mm(const void* const* a, const void* const* b, const void* const* d, const void* const* d2,
                              void* const* out, int32_t m, int32_t count, float alpha, float beta, float beta2,
                              int32_t variant, dmuon_stream_t stream_) {
  DMUON_LOCK;
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
  L.epi_warps = cfg.epi_warps;
  L.alpha = alpha;
  L.beta = beta;
  L.beta2 = beta2;
  L.grid = current_sms();
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

// c_{s,b} of PAPER.md:194: the measured time of the owner-local Muon update of one batch of `batch` matrices of one shape,
// through the complete path the runtime selects (bucketing, tuned tile configurations, block schedule, fused epilogue).
// Runs on scratch buffers of its own (the step is in place: never timed on user data).
DMUON_API int dmuon_measure_cost(int32_t rows, int32_t cols, int32_t batch, int32_t reps, float* ms_out,
                                 dmuon_stream_t stream_) {
  DMUON_LOCK;
  cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
  if (rows <= 0 || cols <= 0 || batch <= 0 || reps <= 0 || !ms_out) { set_error("dmuon_measure_cost: bad arguments"); return DMUON_ERR_INVALID_ARG; }
  int rc = check_device();
  if (rc) return rc;
  const size_t bytes = (static_cast<size_t>(rows) * cols * 2 + 255) / 256 * 256;
  uint8_t* buf = nullptr;
  cudaError_t e = cudaMalloc(&buf, 3 * bytes * batch);
  if (e != cudaSuccess) { cudaGetLastError(); set_error("dmuon_measure_cost: scratch allocation of %zu bytes failed", 3 * bytes * batch); return DMUON_ERR_OOM; }
  std::vector<void*> w(batch), m(batch);
  std::vector<const void*> g(batch);
  std::vector<int32_t> shapes(2 * batch);
  for (int i = 0; i < batch; ++i) {
    w[i] = buf + (3 * i) * bytes;
    g[i] = buf + (3 * i + 1) * bytes;
    m[i] = buf + (3 * i + 2) * bytes;
    shapes[2 * i] = rows;
    shapes[2 * i + 1] = cols;
  }
  // gradient-sized bf16 noise in all three (W, G, M): cost is data independent except for the power the operands draw
  rc = launch_fill_scratch(buf, 3 * bytes * batch, stream);
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (!rc && (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess)) { set_error("dmuon_measure_cost: event creation failed"); rc = DMUON_ERR_CUDA; }
  for (int r = 0; r < 2 && !rc; ++r) rc = muon_step_device(w.data(), g.data(), m.data(), shapes.data(), batch, 0.02f, 0.95f, 0.01f, stream, nullptr);
  if (!rc) {
    cudaEventRecord(e0, stream);
    for (int r = 0; r < reps && !rc; ++r) rc = muon_step_device(w.data(), g.data(), m.data(), shapes.data(), batch, 0.02f, 0.95f, 0.01f, stream, nullptr);
    cudaEventRecord(e1, stream);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaGetLastError(); set_error("dmuon_measure_cost: step failed"); rc = rc ? rc : DMUON_ERR_CUDA; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    *ms_out = ms / reps;
  }
  cudaDeviceSynchronize();
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  cudaFree(buf);
  g_last_plan = 0;      // the workspace now holds the NS results of noise: dmuon_read_ns_output must not hand them out
  return rc;
}

// Owner assignment (Eq. 5): x[s, b, r] batches of configuration (s, b) on rank r minimising the
// largest per-rank sum of measured costs.  mode 0: greedy (longest processing time first); 1: exact branch and bound;
// -1: exact when the number of decision variables is at most `threshold` (S_thr of PAPER.md:206), else greedy.
DMUON_API int dmuon_assign_owners(const int32_t* counts, const int32_t* num_batches, const int32_t* batch_sizes,
                                  const double* costs, int32_t num_shapes, int32_t num_ranks, int32_t mode,
                                  int32_t threshold, int32_t* x_out, double* makespan_out) {
  DMUON_LOCK;
  if (num_shapes < 0 || num_ranks <= 0 || (num_shapes > 0 && (!counts || !num_batches || !batch_sizes || !costs)) || !x_out || !makespan_out) {
    set_error("dmuon_assign_owners: bad arguments");
    return DMUON_ERR_INVALID_ARG;
  }
  long long vars = 0;
  int k = 0;
  for (int s = 0; s < num_shapes; ++s) {
    if (counts[s] < 0 || num_batches[s] <= 0) { set_error("dmuon_assign_owners: shape %d has a bad count or no batch size", s); return DMUON_ERR_INVALID_ARG; }
    bool has_one = false;
    for (int b = 0; b < num_batches[s]; ++b, ++k) {
      if (batch_sizes[k] <= 0 || !(costs[k] >= 0.0)) { set_error("dmuon_assign_owners: shape %d has a bad batch size or cost", s); return DMUON_ERR_INVALID_ARG; }
      has_one = has_one || batch_sizes[k] == 1;
    }
    if (!has_one && counts[s] > 0) {
      // sum_b b x = n_s must be solvable for every residue: require batch size 1 among the candidates
      set_error("dmuon_assign_owners: shape %d needs batch size 1 among its candidates", s);
      return DMUON_ERR_INVALID_ARG;
    }
    vars += static_cast<long long>(num_batches[s]) * num_ranks;
  }
  AssignInput in{num_shapes, num_ranks, counts, num_batches, batch_sizes, costs};
  const bool exact = mode == 1 || (mode == -1 && vars <= threshold);
  if (exact) {
    int rc = assign_owners_exact(in, x_out, makespan_out, 20000000LL);
    if (rc == DMUON_OK) return 1;                    // 1 = exact optimum proven
  }
  int rc = assign_owners_greedy(in, x_out, makespan_out);
  return rc;                                         // 0 = greedy
}

DMUON_API void dmuon_shutdown(void) {
  DMUON_LOCK;
  cudaDeviceSynchronize();
  cudaGetLastError();
  fold_profile();
  g_host.release();
  drop_plans();
  release_workspaces();
  forget_tune_cache();
  g_last_plan = 0;
  if (g_gemm_call.d_probs) cudaFree(g_gemm_call.d_probs);
  if (g_gemm_call.d_units) cudaFree(g_gemm_call.d_units);
  g_gemm_call = GemmCall();
  g_adam_call.release();
  release_pinned();
  for (cudaEvent_t e : g_event_pool) cudaEventDestroy(e);
  g_event_pool.clear();
  g_prof_acc.clear();
  g_launches = 0;
  cudaGetLastError();
}

}  // extern "C"
