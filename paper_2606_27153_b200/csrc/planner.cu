// Host-side planner: buckets, workspace layout, TMA descriptors, grouped-launch tables, autotune + persistent cache.
// See planner.h.  (PAPER.md:180 batching by shape; PAPER.md:184 autotuner and persistent kernel cache.)
#include "planner.h"

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <fstream>
#include <sstream>
#include <sys/stat.h>

#ifndef DMUON_BUILD_ID
#define DMUON_BUILD_ID "dev"      // build.py passes a hash of csrc/: a new build never trusts an old build's timings
#endif

namespace dmuon {

// Gram blocks replace 2 (L - 1) of the m x n products of L steps by 4 (L - 1) m x m products: worth it when the matrix
// is wide.  Tiny Gram matrices (one block) stay on the plain iteration (latency-bound either way).
bool gram_eligible(int m_pad, int n_pad, bool fp32) { return !fp32 && m_pad >= 2 * kBlk && 2 * n_pad >= 3 * m_pad; }

namespace {

constexpr size_t kMaxPlans = 8;              // least-recently-used plans beyond this are dropped
std::vector<std::unique_ptr<Plan>> g_plans;
uint64_t g_stamp = 0;
std::map<std::string, int> g_tune_cache;     // "build op kind m n countbucket" -> variant
bool g_tune_loaded = false;
std::string g_tune_loaded_path;

// One grow-only workspace per device, used by every plan of that device (calls are stream-ordered and buckets run one
// after the other, so nothing needs two regions at a time).
struct DeviceWs {
  uint8_t* ptr = nullptr;
  size_t bytes = 0;
};
DeviceWs g_ws[kMaxDevices];

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
inline int pad128(int v) { return (v + kBlk - 1) / kBlk * kBlk; }
inline int ceil_log2(double v) { int e = 0; while (std::ldexp(1.0, e) < v) ++e; return e; }

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn g_encode = nullptr;

int load_encode() {
  if (g_encode) return DMUON_OK;
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  cudaError_t e = cudaGetDriverEntryPointByVersion("cuTensorMapEncodeTiled", &fn, 12000, cudaEnableDefault, &qres);
  if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn) {
    set_error("cuTensorMapEncodeTiled is not available from the driver (%s)", cudaGetErrorString(e));
    return DMUON_ERR_CUDA;
  }
  g_encode = reinterpret_cast<EncodeTiledFn>(fn);
  return DMUON_OK;
}

template <typename T>
int dev_alloc(Plan& p, T** out, size_t count) {
  void* ptr = nullptr;
  cudaError_t e = cudaMalloc(&ptr, std::max<size_t>(count, 1) * sizeof(T));
  if (e != cudaSuccess) {
    cudaGetLastError();
    set_error("cudaMalloc of %zu bytes failed: %s", count * sizeof(T), cudaGetErrorString(e));
    return DMUON_ERR_OOM;
  }
  p.d_allocs.push_back(ptr);
  *out = static_cast<T*>(ptr);
  return DMUON_OK;
}

template <typename T>
int upload(Plan& p, T** out, const std::vector<T>& host) {
  int rc = dev_alloc(p, out, host.size());
  if (rc) return rc;
  if (!host.empty()) DMUON_CUDA_CHECK(cudaMemcpy(*out, host.data(), host.size() * sizeof(T), cudaMemcpyHostToDevice));
  return DMUON_OK;
}

// ---------------------------------------------------------------------------------------------- layout (host only)
struct Layout {
  std::vector<MatrixInfo> mats;
  std::vector<ShapeTables> shapes;          // layout fields only
  std::vector<std::vector<int>> members;    // matrices of each shape, caller order
  std::vector<BucketPlan> buckets;          // execution order; mats / rec0 / shape / work filled
  size_t ws_bytes = 0;
};

void describe(const int32_t* shapes, int count, bool fp32, bool keep_o, size_t chunk_bytes, Layout& L) {
  const size_t es = fp32 ? 4 : 2;
  L.mats.resize(count);
  std::map<std::tuple<int, int, int>, int> shape_of;
  for (int i = 0; i < count; ++i) {
    MatrixInfo& mi = L.mats[i];
    mi.rows = shapes[2 * i];
    mi.cols = shapes[2 * i + 1];
    mi.m = std::min(mi.rows, mi.cols);               // the Gram matrix is the small one
    mi.n = std::max(mi.rows, mi.cols);
    mi.m_pad = pad128(mi.m);
    mi.n_pad = pad128(mi.n);
    const bool aligned = !fp32 && mi.rows % kBlk == 0 && mi.cols % kBlk == 0;
    mi.kind = !aligned ? K_GENERIC : (mi.rows <= mi.cols ? K_WIDE : K_TALL);
    mi.transposed = mi.kind == K_GENERIC && mi.rows > mi.cols;
    mi.buf_rows = mi.kind == K_GENERIC ? mi.m_pad : mi.rows;
    mi.buf_cols = mi.kind == K_GENERIC ? mi.n_pad : mi.cols;
    mi.gram = gram_eligible(mi.m_pad, mi.n_pad, fp32);
    // fp16 range: entries of the normalised X0 are ~1 / sqrt(m n), those of G0 ~1 / m, both near or below fp16's
    // smallest normal (6.1e-5) for the large shapes; ||X||_2 <= 1.21 and ||G||_2 <= 1.45 bound the other end
    mi.xscale = fp32 ? 1.f : std::ldexp(1.f, std::min(10, std::max(0, ceil_log2(std::sqrt(double(mi.m_pad) * mi.n_pad)) - 4)));
    mi.gscale = fp32 ? 1.f : std::ldexp(1.f, std::min(10, std::max(0, ceil_log2(mi.m_pad) - 2)));
    auto key = std::make_tuple(mi.m_pad, mi.n_pad, mi.kind);
    auto it = shape_of.find(key);
    if (it == shape_of.end()) {
      it = shape_of.emplace(key, static_cast<int>(L.shapes.size())).first;
      ShapeTables st;
      st.m_pad = mi.m_pad; st.n_pad = mi.n_pad; st.kind = mi.kind; st.gram = mi.gram;
      st.buf_rows = mi.buf_rows; st.buf_cols = mi.buf_cols;
      st.xscale = mi.xscale; st.gscale = mi.gscale;
      st.onchip = !fp32 && mi.m_pad == kSmallEdge && mi.n_pad == kSmallEdge && mi.buf_rows == kSmallEdge && mi.buf_cols == kSmallEdge;
      const size_t xb = align_up(static_cast<size_t>(mi.buf_rows) * mi.buf_cols * es, 1024);
      const size_t ab = align_up(static_cast<size_t>(mi.m_pad) * mi.m_pad * es, 1024);
      const int nsq = mi.gram ? 5 : 2;
      st.off_p = 0; st.off_q = xb;
      for (int k = 0; k < 5; ++k) st.off_sq[k] = 2 * xb + std::min(k, nsq - 1) * ab;
      st.mat_bytes = 2 * xb + nsq * ab;
      L.shapes.push_back(st);
      L.members.emplace_back();
    }
    L.members[it->second].push_back(i);
  }
  // chunks: a bucket uses at most chunk_bytes of workspace (keep_o: every matrix keeps its own slot)
  size_t off = 0;
  for (size_t s = 0; s < L.shapes.size(); ++s) {
    ShapeTables& st = L.shapes[s];
    const int n = static_cast<int>(L.members[s].size());
    int slots = n;
    if (!keep_o) {
      const size_t fit = std::max<size_t>(1, chunk_bytes / st.mat_bytes);
      const int chunks = static_cast<int>((n + fit - 1) / fit);
      slots = (n + chunks - 1) / chunks;
    }
    st.slots = slots;
    st.base = keep_o ? off : 0;
    off += static_cast<size_t>(slots) * st.mat_bytes;
    L.ws_bytes = keep_o ? off : std::max(L.ws_bytes, static_cast<size_t>(slots) * st.mat_bytes);
    for (int b0 = 0; b0 < n; b0 += slots) {
      BucketPlan bp;
      bp.shape = static_cast<int>(s);
      bp.mats.assign(L.members[s].begin() + b0, L.members[s].begin() + std::min(n, b0 + slots));
      bp.work = static_cast<double>(bp.mats.size()) * st.m_pad * st.m_pad * (2.0 * st.n_pad + st.m_pad);
      L.buckets.push_back(bp);
    }
  }
  // execution order: most NS work first (stable: chunks of one shape stay together and in caller order)
  std::stable_sort(L.buckets.begin(), L.buckets.end(), [&](const BucketPlan& a, const BucketPlan& b) {
    const double wa = a.work / a.mats.size(), wb = b.work / b.mats.size();      // per matrix: chunks of a shape tie
    return wa > wb;
  });
  int rec = 0;
  for (size_t b = 0; b < L.buckets.size(); ++b) {
    BucketPlan& bp = L.buckets[b];
    bp.rec0 = rec;
    for (size_t k = 0; k < bp.mats.size(); ++k) {
      MatrixInfo& mi = L.mats[bp.mats[k]];
      mi.bucket = static_cast<int>(b);
      mi.slot = static_cast<int>(k);
      mi.rec = rec++;
    }
  }
}

std::string resolve_cache_path(const Options& opt) {
  if (opt.cache_path_set) return opt.cache_path;
  if (const char* e = getenv("DMUON_CACHE")) return e;
  if (const char* h = getenv("HOME")) return std::string(h) + "/.cache/dmuon/tune.txt";
  return "";
}

// File format: one line per entry, "v5 <build> <op> <kind> <m> <n> <countbucket> <variant>".
void load_tune_cache(const std::string& path) {
  if (g_tune_loaded && g_tune_loaded_path == path) return;
  g_tune_cache.clear();
  g_tune_loaded = true;
  g_tune_loaded_path = path;
  if (path.empty()) return;
  std::ifstream in(path);
  std::string line;
  while (std::getline(in, line)) {
    std::istringstream ss(line);
    std::string tag, build;
    int op, kind, m, n, cb, variant;
    if (ss >> tag >> build >> op >> kind >> m >> n >> cb >> variant && tag == "v5" && variant >= 0 && variant < kNumVariants) {
      char key[160];
      snprintf(key, sizeof key, "%s %d %d %d %d %d", build.c_str(), op, kind, m, n, cb);
      g_tune_cache[key] = variant;
    }
  }
}

void save_tune_cache(const std::string& path) {
  if (path.empty()) return;
  const size_t slash = path.find_last_of('/');
  if (slash != std::string::npos) {
    std::string dir = path.substr(0, slash);
    for (size_t i = 1; i <= dir.size(); ++i)
      if (i == dir.size() || dir[i] == '/') mkdir(dir.substr(0, i).c_str(), 0755);
  }
  std::ofstream out(path, std::ios::trunc);
  for (auto& kv : g_tune_cache) out << "v5 " << kv.first << " " << kv.second << "\n";
}

// tiling op (unit table / variant slot) of a product: 0 = the Gram product, 1 = the m x m products, 2 = the X update
inline int tiling_op(GemmOp op) {
  switch (op) {
    case OP_SYRK: case OP_SYRK_T: return 0;
    case OP_SQ: case OP_SQ2: return 1;
    default: return 2;
  }
}
inline GemmOp gram_op(int kind) { return kind == K_TALL ? OP_SYRK_T : OP_SYRK; }
inline GemmOp xupd_op(int kind) { return kind == K_TALL ? OP_XB : OP_BX; }
// extent of an op's output in 128-blocks for a bucket shape
inline void out_blocks(const ShapeTables& st, GemmOp op, int* mb, int* nb) {
  *mb = st.m_pad / kBlk;
  *nb = st.m_pad / kBlk;
  if (op == OP_BX) *nb = st.n_pad / kBlk;
  if (op == OP_XB) *mb = st.n_pad / kBlk;
}

int shape_launch(const Plan& plan, const ShapeTables& st, int count, int rec0, GemmOp op, const GemmProblem* probs,
                 float alpha, float beta, float beta2, const FinalEpilogue& fin, cudaStream_t stream,
                 const TileUnit* units_override = nullptr, int upp_override = 0, int variant_override = -1) {
  const int top = tiling_op(op);
  const TileConfig cfg = variant_config(variant_override >= 0 ? variant_override : st.variant[top]);
  GemmLaunch L;
  L.op = op;
  L.epi = fin.epi;
  L.problems = probs;
  L.units = units_override ? units_override : st.units[top];
  L.recs = plan.d_recs;
  L.units_per_problem = units_override ? upp_override : st.units_per_problem[top];
  L.num_problems = count;
  L.k_blocks = (top == 0 ? st.n_pad : st.m_pad) / kBlkK;
  out_blocks(st, op, &L.m_blocks, &L.n_blocks);
  L.pair = cfg.pair;
  L.epi_warps = cfg.epi_warps;
  L.alpha = alpha;
  L.beta = beta;
  L.beta2 = beta2;
  L.lr = fin.lr;
  L.lrwd = fin.lrwd;
  L.store_c = fin.store_c;
  L.rec_base = rec0;
  L.grid = plan.sm_count;
  return launch_ns_gemm(L, stream);
}

int count_bucket(int count) { return ceil_log2(std::max(1, count)); }

// Time each variant of each tiling op of a bucket shape on the plan's own (scratch-filled) workspace and keep the
// fastest.  Each candidate runs back to back for opt.tune_ms: a handful of isolated launches at boost clock flatter the
// configurations that move more bytes per FLOP, the step itself runs at the power cap ("benchmarked on
// the target hardware").
int autotune_shape(Plan& plan, ShapeTables& st, const Options& opt, cudaStream_t stream, bool* scratch_ready) {
  const std::string path = resolve_cache_path(opt);
  load_tune_cache(path);
  bool dirty = false;
  const GemmOp ops[3] = {gram_op(st.kind), OP_SQ, xupd_op(st.kind)};
  for (int t = 0; t < 3; ++t) {
    const GemmOp op = ops[t];
    char key[160];
    snprintf(key, sizeof key, "%s %d %d %d %d %d", DMUON_BUILD_ID, static_cast<int>(op), st.kind, st.m_pad, st.n_pad,
             count_bucket(st.slots));
    auto it = g_tune_cache.find(key);
    // Unit order of the X update when X does not fit the L2 (126 MB, two halves): the order in which consecutive units
    // share the tile of the LARGE operand reads X once; the other one re-reads all of X for every block of the m x m
    // factor (measured on the 14336 x 4096 bucket: 51.8 GB per launch against 8.6 GB algorithmic, profiles/
    // r2_step_ncu.md).  Isolated timings cannot see that (the products are power-bound either way), so the wasteful
    // order is not a candidate: X' = R X (wide) walks column panels of X, Y' = Y R (tall) walks row blocks of Y.
    const bool general = op == OP_BX || op == OP_XB;
    // (only when the m x m factor itself can stay resident: for 8192 x 8192 both operands stream and timing decides)
    const bool x_exceeds_l2 = general && static_cast<size_t>(st.buf_rows) * st.buf_cols * 2 > (48u << 20) &&
                              static_cast<size_t>(st.m_pad) * st.m_pad * 2 <= (48u << 20);
    const int good_order = op == OP_XB ? 1 : 0;
    int best = st.m_pad >= 2 * kBlk ? 4 : 0;         // untuned default: CTA pair unless the Gram matrix is one block
    if (x_exceeds_l2) best = 4 + good_order;
    if (opt.force_variant[t] >= 0 && variant_valid(op, opt.force_variant[t])) {
      best = opt.force_variant[t];
    } else if (it != g_tune_cache.end() && variant_valid(op, it->second)) {
      best = it->second;
    } else if (opt.autotune) {
      const auto wall0 = std::chrono::steady_clock::now();
      if (!*scratch_ready) {
        int rc = launch_fill_scratch(plan.ws, plan.ws_bytes, stream);
        if (rc) return rc;
        *scratch_ready = true;
      }
      cudaEvent_t e0, e1;
      DMUON_CUDA_CHECK(cudaEventCreate(&e0));
      DMUON_CUDA_CHECK(cudaEventCreate(&e1));
      int mb, nb;
      out_blocks(st, op, &mb, &nb);
      int rc = DMUON_OK;
      struct Cand { int v; TileUnit* du; int n; float ms; };
      std::vector<Cand> cands;
      for (int v = 0; v < kNumVariants && rc == DMUON_OK; ++v) {
        if (!variant_valid(op, v)) continue;
        if (x_exceeds_l2 && variant_config(v).order != good_order) continue;
        std::vector<TileUnit> hu = make_units(op, mb, nb, variant_config(v));
        Cand c{v, nullptr, static_cast<int>(hu.size()), 1e30f};
        if (cudaMalloc(&c.du, hu.size() * sizeof(TileUnit)) != cudaSuccess ||
            cudaMemcpy(c.du, hu.data(), hu.size() * sizeof(TileUnit), cudaMemcpyHostToDevice) != cudaSuccess) rc = DMUON_ERR_CUDA;
        cands.push_back(c);
      }
      // back-to-back launches of one candidate for about `ms_target`; returns the mean launch time
      auto run = [&](const Cand& c, float ms_target, float* mean) {
        float one = 0.f;
        for (int pass = 0; pass < 2 && rc == DMUON_OK; ++pass) {
          const int reps = pass == 0 ? 1 : std::max(2, std::min(4000, static_cast<int>(ms_target / std::max(one, 1e-3f))));
          cudaEventRecord(e0, stream);
          for (int r = 0; r < reps && rc == DMUON_OK; ++r)
            rc = shape_launch(plan, st, st.slots, 0, op, st.tune_probs[t], 1.f, 0.f, 0.f, FinalEpilogue(), stream, c.du, c.n, c.v);
          cudaEventRecord(e1, stream);
          if (cudaEventSynchronize(e1) != cudaSuccess) rc = DMUON_ERR_CUDA;
          float total = 0.f;
          cudaEventElapsedTime(&total, e0, e1);
          one = total / reps;
        }
        *mean = one;
      };
      // 1. bring the board to the state the step runs in: a few candidates' worth of back-to-back launches of the default
      //    configuration (a cold board at boost clock flatters whichever candidate runs first)
      float burn = 0.f;
      for (const Cand& c : cands)
        if (c.v == best) run(c, 4.f * opt.tune_ms, &burn);
      // 2. every candidate for tune_ms
      for (Cand& c : cands) {
        run(c, opt.tune_ms, &c.ms);
        if (getenv("DMUON_LOG")) fprintf(stderr, "[dmuon] tune op %d kind %d %dx%d x%d variant %d: %.4f ms\n", static_cast<int>(op), st.kind, st.m_pad, st.n_pad, st.slots, c.v, c.ms);
      }
      // 3. the two fastest once more, alternating, and the decision on the sum of both rounds
      std::sort(cands.begin(), cands.end(), [](const Cand& a, const Cand& b) { return a.ms < b.ms; });
      if (cands.size() >= 2 && rc == DMUON_OK) {
        float again[2] = {0.f, 0.f};
        for (int round = 0; round < 2; ++round)
          for (int k = 0; k < 2; ++k) {
            float ms = 0.f;
            run(cands[k], 0.5f * opt.tune_ms, &ms);
            again[k] += 0.5f * ms;
          }
        cands[0].ms = 0.5f * (cands[0].ms + again[0]);
        cands[1].ms = 0.5f * (cands[1].ms + again[1]);
        if (getenv("DMUON_LOG")) fprintf(stderr, "[dmuon] tune op %d: finalists %d (%.4f ms) and %d (%.4f ms)\n", static_cast<int>(op), cands[0].v, cands[0].ms, cands[1].v, cands[1].ms);
        // a tie within 1 % goes to the lower variant number, so that two runs agree
        if (cands[1].ms < cands[0].ms * (cands[1].v < cands[0].v ? 1.01f : 0.99f)) std::swap(cands[0], cands[1]);
      }
      for (Cand& c : cands) cudaFree(c.du);
      if (rc) { cudaEventDestroy(e0); cudaEventDestroy(e1); set_error("autotune launch failed"); return rc; }
      if (!cands.empty()) best = cands[0].v;
      cudaEventDestroy(e0);
      cudaEventDestroy(e1);
      g_tune_cache[key] = best;
      dirty = true;
      st.tuned_now = true;
      plan.tune_seconds += std::chrono::duration<double>(std::chrono::steady_clock::now() - wall0).count();
    }
    st.variant[t] = best;
  }
  if (dirty) save_tune_cache(path);
  return DMUON_OK;
}

void drop_plans_of_device(int device, bool shared_ws_only) {
  for (size_t i = 0; i < g_plans.size();) {
    if (g_plans[i]->device == device && (!shared_ws_only || !g_plans[i]->ext_ws)) g_plans.erase(g_plans.begin() + i);
    else ++i;
  }
}

}  // namespace

int tune_cache_entries() { return static_cast<int>(g_tune_cache.size()); }

void forget_tune_cache() {       // the in-memory copy; the file stays
  g_tune_cache.clear();
  g_tune_loaded = false;
  g_tune_loaded_path.clear();
}

int fill_problem(GemmProblem& g, GemmOp op, const void* a_mat, uint64_t a_rows, uint64_t a_cols, const void* b_mat,
                 uint64_t b_rows, uint64_t b_cols, const void* d, void* c, int ldc, const void* d2, int rec) {
  memset(&g, 0, sizeof g);
  int rc;
  if (op == OP_SYRK_T) rc = encode_tmap_2d(&g.tmA, a_mat, a_rows, a_cols, 64, kBlkK);   // MN-major: 64 (m) x 64 (k) boxes
  else rc = encode_tmap_2d(&g.tmA, a_mat, a_rows, a_cols, kBlkK, kBlk);
  if (rc) return rc;
  if (op == OP_BX || op == OP_SYRK_T) rc = encode_tmap_2d(&g.tmB, b_mat, b_rows, b_cols, 64, kBlkK);   // MN-major: 64 (n) x 64 (k) boxes
  else rc = encode_tmap_2d(&g.tmB, b_mat, b_rows, b_cols, kBlkK, kBlk);
  if (rc) return rc;
  // epilogue tiles: C, D, D2 share one shape (rows x ldc); 32 x 32 boxes with the 64-byte swizzle
  const uint64_t c_rows = (op == OP_BX || op == OP_XB) ? a_rows : static_cast<uint64_t>(ldc);
  if (c && (rc = encode_tmap_2d(&g.tmC, c, c_rows, ldc, 32, 32, CU_TENSOR_MAP_SWIZZLE_64B))) return rc;
  if (d && (rc = encode_tmap_2d(&g.tmD, d, c_rows, ldc, 32, 32, CU_TENSOR_MAP_SWIZZLE_64B))) return rc;
  if (d2 && (rc = encode_tmap_2d(&g.tmD2, d2, c_rows, ldc, 32, 32, CU_TENSOR_MAP_SWIZZLE_64B))) return rc;
  g.ldc = ldc;
  g.rec = rec;
  return DMUON_OK;
}

Plan::~Plan() {
  int cur = 0;
  cudaGetDevice(&cur);
  if (cur != device) cudaSetDevice(device);
  for (void* p : d_allocs) cudaFree(p);
  if (cur != device) cudaSetDevice(cur);
}

TileConfig variant_config(int variant) {
  TileConfig c;
  if (variant >= 4) {
    c.pair = true;
    c.order = variant & 1;
    c.epi_warps = variant >= 6 ? 8 : 4;
  } else {
    c.width = (variant & 1) ? 1 : 2;
    c.order = (variant >> 1) & 1;
  }
  return c;
}

bool variant_valid(GemmOp op, int variant) {
  if (variant < 0 || variant >= kNumVariants) return false;
  return op == OP_BX || op == OP_XB || variant_config(variant).order == 0;   // symmetric ops have one ordering
}

std::vector<TileUnit> make_units(GemmOp op, int mb, int nb, const TileConfig& cfg) {
  std::vector<TileUnit> u;
  auto push = [&](int i, int j, int w) { u.push_back(TileUnit{static_cast<int16_t>(i), static_cast<int16_t>(j), static_cast<int16_t>(w), 0}); };
  const bool general = op == OP_BX || op == OP_XB;
  if (cfg.pair) {
    // 256 x 256 units; an odd block count leaves a half-empty last unit (operands zero-filled, stores skipped)
    const int MB = (mb + 1) / 2, NB = (nb + 1) / 2;
    if (general) {
      if (cfg.order == 0) { for (int j = 0; j < NB; ++j) for (int i = 0; i < MB; ++i) push(i, j, 2); }
      else                { for (int i = 0; i < MB; ++i) for (int j = 0; j < NB; ++j) push(i, j, 2); }
    } else {
      for (int i = 0; i < MB; ++i) for (int j = i; j < MB; ++j) push(i, j, 2);
    }
    return u;
  }
  if (general) {
    if (cfg.order == 0) {
      for (int j = 0; j < nb; j += cfg.width)
        for (int i = 0; i < mb; ++i) push(i, j, std::min(cfg.width, nb - j));
    } else {
      for (int i = 0; i < mb; ++i)
        for (int j = 0; j < nb; j += cfg.width) push(i, j, std::min(cfg.width, nb - j));
    }
  } else {
    // upper-triangular blocks only (PAPER.md:182 computes one triangle and reconstructs the other in the epilogue)
    for (int i = 0; i < mb; ++i)
      for (int j = i; j < mb; j += cfg.width) push(i, j, std::min(cfg.width, mb - j));
  }
  return u;
}

int encode_tmap_2d(CUtensorMap* out, const void* base, uint64_t rows, uint64_t cols, uint32_t box_cols,
                   uint32_t box_rows, CUtensorMapSwizzle swizzle) {
  int rc = load_encode();
  if (rc) return rc;
  const cuuint64_t gdim[2] = {cols, rows};
  const cuuint64_t gstride[1] = {cols * sizeof(__half)};
  const cuuint32_t box[2] = {box_cols, box_rows};
  const cuuint32_t estr[2] = {1, 1};
  CUresult r = g_encode(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, const_cast<void*>(base), gdim, gstride, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, swizzle, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    set_error("cuTensorMapEncodeTiled failed (%d) for %llu x %llu, box %u x %u, base %p", static_cast<int>(r),
              static_cast<unsigned long long>(rows), static_cast<unsigned long long>(cols), box_rows, box_cols, base);
    return DMUON_ERR_CUDA;
  }
  return DMUON_OK;
}

// {cols, rows, slots} over `slots` row-major fp16 matrices `slot_bytes` apart; box {box_cols, box_rows, 1}.
int encode_tmap_3d(CUtensorMap* out, const void* base, uint64_t rows, uint64_t cols, uint64_t slots, uint64_t slot_bytes,
                   uint32_t box_cols, uint32_t box_rows) {
  int rc = load_encode();
  if (rc) return rc;
  const cuuint64_t gdim[3] = {cols, rows, slots};
  const cuuint64_t gstride[2] = {cols * sizeof(__half), slot_bytes};
  const cuuint32_t box[3] = {box_cols, box_rows, 1};
  const cuuint32_t estr[3] = {1, 1, 1};
  CUresult r = g_encode(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 3, const_cast<void*>(base), gdim, gstride, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    set_error("cuTensorMapEncodeTiled (3-D) failed (%d) for %llu x %llu x %llu, slot stride %llu", static_cast<int>(r),
              static_cast<unsigned long long>(rows), static_cast<unsigned long long>(cols),
              static_cast<unsigned long long>(slots), static_cast<unsigned long long>(slot_bytes));
    return DMUON_ERR_CUDA;
  }
  return DMUON_OK;
}

int check_device() {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) {
    cudaGetLastError();
    set_error("no CUDA device: %s", cudaGetErrorString(e));
    return DMUON_ERR_UNSUPPORTED_DEVICE;
  }
  int major = 0;
  e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
  if (e != cudaSuccess || major != 10) {
    cudaGetLastError();
    set_error("libdmuon needs an sm_100 (B200) device; found compute capability major %d", major);
    return DMUON_ERR_UNSUPPORTED_DEVICE;
  }
  if (dev >= kMaxDevices) {
    set_error("device ordinal %d is not supported (max %d)", dev, kMaxDevices - 1);
    return DMUON_ERR_UNSUPPORTED_DEVICE;
  }
  return DMUON_OK;
}

size_t plan_workspace_bytes(const int32_t* shapes, int count, const Options& opt) {
  Layout L;
  describe(shapes, count, opt.fp32_check, opt.keep_o, opt.chunk_bytes, L);
  return L.ws_bytes;
}

void drop_plans() { g_plans.clear(); }

int captured_plans() {
  int n = 0;
  for (auto& up : g_plans) n += up->captured ? 1 : 0;
  return n;
}

void forget_captures() {
  for (auto& up : g_plans) up->captured = false;
}

Plan* find_plan(uint64_t id) {
  for (auto& up : g_plans)
    if (up->id == id) return up.get();
  return nullptr;
}

void release_workspaces() {
  int cur = 0;
  if (cudaGetDevice(&cur) != cudaSuccess) { cudaGetLastError(); return; }
  for (int d = 0; d < kMaxDevices; ++d) {
    if (!g_ws[d].ptr) continue;
    cudaSetDevice(d);
    cudaFree(g_ws[d].ptr);
    g_ws[d] = DeviceWs();
  }
  cudaSetDevice(cur);
  cudaGetLastError();
}

int get_plan(const int32_t* shapes, int count, const Options& opt, void* ext_ws, size_t ext_bytes, cudaStream_t stream,
             Plan** out) {
  int rc = check_device();
  if (rc) return rc;
  int dev = 0;
  cudaGetDevice(&dev);
  for (auto& up : g_plans) {
    Plan& p = *up;
    if (p.device == dev && p.fp32 == opt.fp32_check && p.keep_o == opt.keep_o && p.chunk_bytes == opt.chunk_bytes &&
        p.ext_ws == ext_ws && p.shapes.size() == static_cast<size_t>(2 * count) &&
        (count == 0 || memcmp(p.shapes.data(), shapes, sizeof(int32_t) * 2 * count) == 0)) {
      p.stamp = ++g_stamp;
      *out = &p;
      return DMUON_OK;
    }
  }

  std::unique_ptr<Plan> up(new Plan);
  Plan& p = *up;
  p.shapes.assign(shapes, shapes + 2 * count);
  p.fp32 = opt.fp32_check;
  p.keep_o = opt.keep_o;
  p.chunk_bytes = opt.chunk_bytes;
  p.device = dev;
  p.ext_ws = ext_ws;
  p.stamp = ++g_stamp;
  p.id = p.stamp;
  {
    Layout L;
    describe(shapes, count, p.fp32, p.keep_o, p.chunk_bytes, L);
    p.mats = std::move(L.mats);
    p.shapes_tbl = std::move(L.shapes);
    p.buckets = std::move(L.buckets);
    p.ws_bytes = L.ws_bytes;
  }
  cudaDeviceGetAttribute(&p.sm_count, cudaDevAttrMultiProcessorCount, dev);

  // ---- workspace: the caller's, or the device's shared grow-only region
  if (ext_ws) {
    if (ext_bytes < p.ws_bytes) {
      set_error("caller workspace of %zu bytes is smaller than the %zu bytes this shape set needs", ext_bytes, p.ws_bytes);
      return DMUON_ERR_OOM;
    }
    p.ws = static_cast<uint8_t*>(ext_ws);
  } else {
    DeviceWs& w = g_ws[dev];
    if (w.bytes < p.ws_bytes) {
      // growing moves the region: plans that point into the old one are dropped (their tuned choices stay cached).
      // A captured graph holds raw pointers into the region and into those plans' tables: refuse rather than free them.
      for (auto& q : g_plans)
        if (q->device == dev && !q->ext_ws && q->captured) {
          set_error("this shape set needs a %zu-byte workspace (the device's is %zu) but a captured CUDA graph refers to the "
                    "current one: destroy the graphs and set option graphs_destroyed=1, or size the workspace first with "
                    "dmuon_warmup on the largest shape set before capturing", p.ws_bytes, w.bytes);
          return DMUON_ERR_INVALID_ARG;
        }
      DMUON_CUDA_CHECK(cudaDeviceSynchronize());
      drop_plans_of_device(dev, true);
      if (w.ptr) cudaFree(w.ptr);
      w = DeviceWs();
      void* ptr = nullptr;
      cudaError_t e = cudaMalloc(&ptr, std::max<size_t>(p.ws_bytes, 1));
      if (e != cudaSuccess) {
        cudaGetLastError();
        set_error("cudaMalloc of the %zu-byte workspace failed: %s", p.ws_bytes, cudaGetErrorString(e));
        return DMUON_ERR_OOM;
      }
      w.ptr = static_cast<uint8_t*>(ptr);
      w.bytes = p.ws_bytes;
    }
    p.ws = w.ptr;
  }
  // check mode: padding of the fp32 buffers must be zero (the tensor-core path's padding is written by the normalise kernel
  // for generic matrices and does not exist for aligned ones)
  DMUON_CUDA_CHECK(cudaMemsetAsync(p.ws, 0, p.ws_bytes, stream));
  // building a plan writes the region (this memset, the autotune's noise): NS results another plan left there are gone,
  // whether or not a step follows (dmuon_warmup / dmuon_describe_plan build plans without running one)
  for (auto& q : g_plans)
    if (q->device == dev && q->ws == p.ws) q->o_valid = false;

  // ---- elementwise records and per-bucket work lists
  const size_t nrec = std::max(count, 1);
  p.h_recs.resize(nrec);
  memset(p.h_recs.data(), 0, nrec * sizeof(MatRec));
  for (int i = 0; i < count; ++i) {
    const MatrixInfo& mi = p.mats[i];
    const ShapeTables& st = p.shapes_tbl[p.buckets[mi.bucket].shape];
    uint8_t* slot = p.ws + st.base + static_cast<size_t>(mi.slot) * st.mat_bytes;
    MatRec& r = p.h_recs[mi.rec];
    r.U = slot + st.off_p;
    r.X0 = slot + st.off_q;
    r.O = nullptr;
    r.rows = mi.rows; r.cols = mi.cols;
    r.m_pad = mi.buf_rows; r.n_pad = mi.buf_cols;
    r.transposed = mi.transposed ? 1 : 0;
    r.scale = static_cast<float>(std::sqrt(std::max(1.0, static_cast<double>(mi.rows) / mi.cols)));   // reading N4
    r.xscale = mi.xscale;
    r.inv_xscale = 1.f / mi.xscale;
  }
  if ((rc = dev_alloc(p, &p.d_recs, nrec))) return rc;
  if ((rc = dev_alloc(p, &p.d_inv_norm, nrec))) return rc;
  std::vector<int> mat_of_rec(count, -1);
  for (int i = 0; i < count; ++i) mat_of_rec[p.mats[i].rec] = i;
  for (BucketPlan& bp : p.buckets) {
    // prefix arrays over ALL records: the records outside the bucket have no work items
    std::vector<int64_t> flat_prefix(count + 1, 0), tile_prefix(count + 1, 0), ptile_prefix(count + 1, 0), fa_prefix(count + 1, 0);
    for (int r = 0; r < count; ++r) {
      const MatrixInfo& mi = p.mats[mat_of_rec[r]];
      const bool member = r >= bp.rec0 && r < bp.rec0 + static_cast<int>(bp.mats.size());
      const int64_t elems = static_cast<int64_t>(mi.rows) * mi.cols;
      const bool aligned = mi.kind != K_GENERIC;
      flat_prefix[r + 1] = flat_prefix[r] + (member ? (elems + kFlatChunk - 1) / kFlatChunk : 0);
      fa_prefix[r + 1] = fa_prefix[r] + (member && aligned ? elems / kFlatChunk : 0);
      tile_prefix[r + 1] = tile_prefix[r] + (member && !aligned ? static_cast<int64_t>((mi.rows + kTile - 1) / kTile) * ((mi.cols + kTile - 1) / kTile) : 0);
      ptile_prefix[r + 1] = ptile_prefix[r] + (member && !aligned ? static_cast<int64_t>(mi.m_pad / kTile) * (mi.n_pad / kTile) : 0);
    }
    int64_t *d_flat = nullptr, *d_tile = nullptr, *d_ptile = nullptr, *d_fa = nullptr;
    float* d_partials = nullptr;
    if ((rc = upload(p, &d_flat, flat_prefix))) return rc;
    if ((rc = upload(p, &d_tile, tile_prefix))) return rc;
    if ((rc = upload(p, &d_ptile, ptile_prefix))) return rc;
    if ((rc = upload(p, &d_fa, fa_prefix))) return rc;
    if ((rc = dev_alloc(p, &d_partials, static_cast<size_t>(flat_prefix[count])))) return rc;
    ElemTables& T = bp.tables;
    T.recs = p.d_recs;
    T.flat_prefix = d_flat;
    T.tile_prefix = d_tile;
    T.ptile_prefix = d_ptile;
    T.fa_prefix = d_fa;
    T.count = count;
    T.flat_chunks = flat_prefix[count];
    T.tiles = tile_prefix[count];
    T.ptiles = ptile_prefix[count];
    T.fa_chunks = fa_prefix[count];
    T.partials = d_partials;
    T.inv_norm = p.d_inv_norm;
  }

  // ---- grouped GEMM tables (tensor-core mode only): scratch problems for the autotuner, tile units per op.  The
  //      launch programs of the NS steps are built on first use (build_program), they depend on the step count.
  if (!p.fp32) {
    bool scratch_ready = false;
    for (ShapeTables& st : p.shapes_tbl) {
      if (st.onchip &&
          (rc = encode_tmap_3d(&st.tm_x0, p.ws + st.base + st.off_q, kSmallEdge, kSmallEdge, st.slots, st.mat_bytes, kBlkK, kBlk)))
        return rc;
      // buckets that run in the on-chip kernel need no tile configuration: no scratch tables, nothing to time (if the
      // option is switched off later, the same plan runs the grouped products with the default configuration)
      const bool tune = !(st.onchip && opt.small_fused);
      const size_t nprob = tune ? st.slots : 0;
      std::vector<GemmProblem> tp[3];
      for (int t = 0; t < 3; ++t) tp[t].resize(nprob);
      for (size_t k = 0; k < nprob; ++k) {
        uint8_t* slot = p.ws + st.base + k * st.mat_bytes;
        void* XQ = slot + st.off_q;
        void* XP = slot + st.off_p;
        void* A = slot + st.off_sq[0];
        void* B = slot + st.off_sq[1];
        const uint64_t m = st.m_pad, br = st.buf_rows, bc = st.buf_cols;
        if ((rc = fill_problem(tp[0][k], gram_op(st.kind), XQ, br, bc, XQ, br, bc, nullptr, A, st.m_pad))) return rc;
        if ((rc = fill_problem(tp[1][k], OP_SQ, A, m, m, A, m, m, A, B, st.m_pad))) return rc;
        if (st.kind == K_TALL) rc = fill_problem(tp[2][k], OP_XB, XQ, br, bc, B, m, m, XQ, XP, st.buf_cols);
        else rc = fill_problem(tp[2][k], OP_BX, B, m, m, XQ, br, bc, XQ, XP, st.buf_cols);
        if (rc) return rc;
      }
      for (int t = 0; t < 3; ++t)
        if ((rc = upload(p, &st.tune_probs[t], tp[t]))) return rc;
      // tile configuration: tuned (cache or measurement) or the default
      if (tune) { if ((rc = autotune_shape(p, st, opt, stream, &scratch_ready))) return rc; }
      else for (int t = 0; t < 3; ++t) st.variant[t] = 4;
      const GemmOp ops[3] = {gram_op(st.kind), OP_SQ, xupd_op(st.kind)};
      for (int t = 0; t < 3; ++t) {
        int mb, nb;
        out_blocks(st, ops[t], &mb, &nb);
        std::vector<TileUnit> hu = make_units(ops[t], mb, nb, variant_config(st.variant[t]));
        st.units_per_problem[t] = static_cast<int>(hu.size());
        if ((rc = upload(p, &st.units[t], hu))) return rc;
      }
      if (st.m_pad >= 2 * kBlk) {
        // program kernel: CTA-pair units for every product; the X update in the tuned order (or the one that reads X once)
        for (int t = 0; t < 3; ++t) {
          int mb, nb;
          out_blocks(st, ops[t], &mb, &nb);
          TileConfig cfg;
          cfg.pair = true;
          cfg.order = t == 2 ? variant_config(st.variant[2]).order : 0;
          std::vector<TileUnit> hu = make_units(ops[t], mb, nb, cfg);
          st.prog_upp[t] = static_cast<int>(hu.size());
          if ((rc = upload(p, &st.prog_units[t], hu))) return rc;
        }
        if ((rc = dev_alloc(p, &st.d_done, static_cast<size_t>(st.slots) + 1))) return rc;     // + the unit queue
      }
    }
    if (scratch_ready) DMUON_CUDA_CHECK(cudaMemsetAsync(p.ws, 0, p.ws_bytes, stream));
  }
  DMUON_CUDA_CHECK(cudaDeviceSynchronize());
  // least-recently-used plans make room
  // (never a plan that a captured CUDA graph refers to: its replay reads the plan's device tables)
  while (g_plans.size() >= kMaxPlans) {
    size_t victim = g_plans.size();
    for (size_t i = 0; i < g_plans.size(); ++i)
      if (!g_plans[i]->captured && (victim == g_plans.size() || g_plans[i]->stamp < g_plans[victim]->stamp)) victim = i;
    if (victim == g_plans.size()) {
      set_error("all %zu cached plans are referred to by captured CUDA graphs: destroy the graphs and set option "
                "graphs_destroyed=1", g_plans.size());
      return DMUON_ERR_INVALID_ARG;
    }
    g_plans.erase(g_plans.begin() + victim);
  }
  g_plans.push_back(std::move(up));
  *out = g_plans.back().get();
  return DMUON_OK;
}

std::string partition_key(const Partition& part) {
  std::string k;
  for (int L : part) k += static_cast<char>('0' + L);
  return k;
}

// Block lengths for `steps` NS steps.  A 3-block is taken only as the FIRST block: there ||X||_F = 1 bounds ||G||, so
// the fp16 rounding of G is small in absolute terms; later blocks are 2-blocks (measured).
// A block is shortened until the error gain of its Gram recurrence, prod a_j^2 over all but its last step, is <= 200
// (the default a = 3.4445 gives 11.9 for a 2-block and 140.8 for a 3-block).
Partition choose_partition(int steps, const float* coeffs, bool per_step, bool gram) {
  Partition part;
  int s = 0;
  while (s < steps) {
    const int rem = steps - s;
    int L = 1;
    if (gram) {
      L = (part.empty() && rem >= 3 && rem != 4) ? 3 : (rem >= 2 ? 2 : 1);
      while (L > 1) {
        double gain = 1.0;
        for (int j = s; j < s + L - 1; ++j) {
          const double a = coeffs[per_step ? 3 * j : 0];
          gain *= a * a;
        }
        if (gain <= 200.0) break;   // also false for NaN
        --L;
      }
    }
    part.push_back(L);
    s += L;
  }
  return part;
}

bool bucket_onchip(const Plan& plan, const ShapeTables& st, int steps, const Options& opt) {
  return !plan.fp32 && st.onchip && opt.small_fused && steps >= 1 && steps <= kSmallMaxSteps;
}

size_t program_launches(const Partition& part) {
  size_t n = 0;
  for (int L : part) n += 3 + 4 * static_cast<size_t>(L - 1);
  return n;
}

bool bucket_program(const Plan& plan, const ShapeTables& st, size_t num_launches, const Options& opt) {
  // "auto": where the m x m factors are L2-sized (m >= 2048) the program kernel wins 5-10 % (fewer DRAM bytes, hence
  // more clock under the power cap); below that the per-product launches with their tuned tilings are as fast or faster
  const bool wanted = opt.program == 1 || (opt.program == 2 && st.m_pad >= 2048);
  return !plan.fp32 && wanted && st.d_done && num_launches >= 1 && num_launches <= static_cast<size_t>(kMaxProgPhases);
}

int result_parity(const Plan& plan, const ShapeTables& st, int steps, const float* coeffs, bool per_step, const Options& opt) {
  if (plan.fp32) return steps & 1;
  if (bucket_onchip(plan, st, steps, opt)) return 1;      // reads Q, leaves X_k in P
  return static_cast<int>(choose_partition(steps, coeffs, per_step, st.gram && opt.gram_blocks).size()) & 1;
}

bool bucket_fuses(const Plan& plan, const ShapeTables& st, int steps, const Options& opt) {
  return !plan.fp32 && opt.fuse && st.kind != K_GENERIC && steps > 0;
}

namespace {

// Build the launch list of one bucket shape for a partition of the steps into blocks.  m x m buffers: 0 = G, 1/2 = B
// and B' (alternating), 3 = T, 4 = R.
int build_program(Plan& p, ShapeTables& st, const Partition& part, NsProgram& prog) {
  const size_t nprob = st.slots;
  int rc;
  const bool tall = st.kind == K_TALL;
  // stored-shape tag of the profile names: tall buckets read "rows x cols" of the stored matrices
  const std::string dims = "[" + std::to_string(tall ? st.n_pad : st.m_pad) + "x" + std::to_string(tall ? st.m_pad : st.n_pad) + "]";
  auto emit = [&](GemmOp op, CoefKind ck, int s0, int s1, const char* name, int a_buf, int b_buf, int d_buf, int d2_buf,
                  int c_buf, int xsrc) -> int {
    // buffer ids: 0..4 = m x m buffers; 10 / 11 = X in Q / P
    std::vector<GemmProblem> hp(nprob);
    for (size_t k = 0; k < nprob; ++k) {
      uint8_t* slot = p.ws + st.base + k * st.mat_bytes;
      auto buf = [&](int id) -> void* {
        if (id < 0) return nullptr;
        if (id >= 10) return slot + (id == 10 ? st.off_q : st.off_p);
        return slot + st.off_sq[id];
      };
      const uint64_t m = st.m_pad, br = st.buf_rows, bc = st.buf_cols;
      const int rec = static_cast<int>(k);
      if (op == OP_SYRK || op == OP_SYRK_T) rc = fill_problem(hp[k], op, buf(xsrc), br, bc, buf(xsrc), br, bc, nullptr, buf(c_buf), st.m_pad, nullptr, rec);
      else if (op == OP_BX) rc = fill_problem(hp[k], op, buf(a_buf), m, m, buf(xsrc), br, bc, buf(xsrc), buf(c_buf), st.buf_cols, nullptr, rec);
      else if (op == OP_XB) rc = fill_problem(hp[k], op, buf(xsrc), br, bc, buf(a_buf), m, m, buf(xsrc), buf(c_buf), st.buf_cols, nullptr, rec);
      else rc = fill_problem(hp[k], op, buf(a_buf), m, m, buf(b_buf), m, m, buf(d_buf), buf(c_buf), st.m_pad, buf(d2_buf), rec);
      if (rc) return rc;
    }
    NsLaunch L;
    L.op = op; L.ck = ck; L.s0 = s0; L.s1 = s1;
    L.name = std::string(name) + dims;
    if ((rc = upload(p, &L.probs, hp))) return rc;
    prog.launches.push_back(L);
    return DMUON_OK;
  };
  const GemmOp syrk = gram_op(st.kind), xupd = xupd_op(st.kind);
  const char* syrk_name = tall ? "ns_syrk_xtx" : "ns_syrk_xxt";
  const char* xupd_name = tall ? "ns_xb_update" : "ns_bx_update";
  int s = 0, par = 0;   // X0 is in Q (parity 0)
  for (int L : part) {
    if (L > 1 && !st.gram) { set_error("internal: Gram block on a bucket without Gram buffers"); return DMUON_ERR_INVALID_ARG; }
    if (L > 3) { set_error("internal: Gram block longer than 3"); return DMUON_ERR_INVALID_ARG; }
    const int xs = 10 + par, xd = 10 + (1 - par);
    int g = 0, bc = 1, bn = 2, t = 3, r = 1;     // R_0 = B_0 (alias)
    if ((rc = emit(syrk, CK_GRAM, s, s, syrk_name, -1, -1, -1, -1, g, xs))) return rc;                  // G = X X^T
    if ((rc = emit(OP_SQ, CK_POLY, s, s, "ns_sq_poly", g, g, g, -1, bc, -1))) return rc;                // B = b G + c G G
    for (int i = 1; i < L; ++i) {
      const int stp = s + i;
      if ((rc = emit(OP_SQ, CK_A, stp - 1, stp - 1, "ns_gram_mm", bc, g, g, -1, t, -1))) return rc;     // T = a G + B G
      if ((rc = emit(OP_SQ, CK_A, stp - 1, stp - 1, "ns_gram_mm", t, bc, t, -1, g, -1))) return rc;     // G' = a T + T B
      if ((rc = emit(OP_SQ, CK_POLY, stp, stp, "ns_sq_poly", g, g, g, -1, bn, -1))) return rc;          // B' = b G' + c G' G'
      const int rn = (i == 1) ? 4 : t;            // free buffer: R (i = 1), then T (not needed after G')
      if ((rc = emit(OP_SQ2, CK_RACC, s, stp, "ns_gram_mm", bn, r, bn, r, rn, -1))) return rc;           // R' = (prod a) B' + a R + B' R
      r = rn;
      const int tmp = bc; bc = bn; bn = tmp;
    }
    if ((rc = emit(xupd, CK_APOW, s, s + L - 1, xupd_name, r, -1, -1, -1, xd, xs))) return rc;           // X' = (prod a) X + R X
    s += L;
    par ^= 1;
    ++prog.x_updates;
  }
  return DMUON_OK;
}

void launch_coefs(const NsLaunch& L, const ShapeTables& st, const float* coeffs, bool per_step, float* alpha,
                  float* beta, float* beta2) {
  auto co = [&](int step, int which) { return coeffs[(per_step ? 3 * step : 0) + which]; };
  *alpha = 1.f; *beta = 0.f; *beta2 = 0.f;
  double prod = 1.0;
  const double g = st.gscale, cx = st.xscale;
  switch (L.ck) {
    case CK_GRAM: *alpha = static_cast<float>(g / (cx * cx)); break;
    case CK_POLY: *alpha = static_cast<float>(co(L.s1, 2) / (g * g)); *beta = static_cast<float>(co(L.s1, 1) / g); break;
    case CK_A: *beta = co(L.s1, 0); break;
    case CK_RACC:
      for (int j = L.s0; j < L.s1; ++j) prod *= co(j, 0);
      *beta = static_cast<float>(prod);
      *beta2 = co(L.s1, 0);
      break;
    case CK_APOW:
      for (int j = L.s0; j <= L.s1; ++j) prod *= co(j, 0);
      *beta = static_cast<float>(prod);
      break;
  }
}

}  // namespace

int run_ns_bucket(Plan& plan, int bucket, int steps, const float* coeffs, bool per_step, const Options& opt,
                  const FinalEpilogue& fin, cudaStream_t stream) {
  BucketPlan& bp = plan.buckets[bucket];
  ShapeTables& st = plan.shapes_tbl[bp.shape];
  const int count = static_cast<int>(bp.mats.size());
  if (bucket_onchip(plan, st, steps, opt)) {
    // every step in one launch; the workspace holds c X and the kernel keeps g G on chip (same scales and the same
    // epilogue constants as the grouped products: launch_coefs)
    const bool fused = bucket_fuses(plan, st, steps, opt) && fin.epi != EPI_F16;
    SmallLaunch L;
    L.tmX = &st.tm_x0;
    L.out = plan.ws + st.base + st.off_p;
    L.slot_bytes = st.mat_bytes;
    L.recs = plan.d_recs;
    L.rec_base = bp.rec0;
    L.count = count;
    L.steps = steps;
    const double g = st.gscale, cx = st.xscale;
    L.gram_alpha = static_cast<float>(g / (cx * cx));
    for (int s = 0; s < steps; ++s) {
      const float* q = coeffs + (per_step ? 3 * s : 0);
      L.poly_alpha[s] = static_cast<float>(q[2] / (g * g));
      L.poly_beta[s] = static_cast<float>(q[1] / g);
      L.x_beta[s] = q[0];
    }
    L.epi = fused ? fin.epi : EPI_F16;
    L.lr = fin.lr;
    L.lrwd = fin.lrwd;
    L.store_c = fused ? fin.store_c : true;
    L.grid = plan.sm_count;
    const std::string name = std::string(!fused ? "ns_small_fused" : fin.epi == EPI_BF16 ? "ns_small_fused_out" : "ns_small_fused_apply") + "[" +
                             std::to_string(st.m_pad) + "x" + std::to_string(st.n_pad) + "]";
    ProfScope ps(name.c_str(), stream);
    return launch_ns_small(L, stream);
  }
  if (!plan.fp32) {
    const Partition part = choose_partition(steps, coeffs, per_step, st.gram && opt.gram_blocks);
    const std::string key = partition_key(part);
    auto it = st.programs.find(key);
    if (it == st.programs.end()) {
      NsProgram prog;
      int rc = build_program(plan, st, part, prog);
      if (rc) return rc;
      it = st.programs.emplace(key, std::move(prog)).first;
    }
    const bool fused = bucket_fuses(plan, st, steps, opt) && fin.epi != EPI_F16;
    const size_t nl = it->second.launches.size();
    if (bucket_program(plan, st, nl, opt)) {
      ProgLaunch P;
      P.num_phases = static_cast<int>(nl);
      for (size_t li = 0; li < nl; ++li) {
        const NsLaunch& L = it->second.launches[li];
        P.ph[li].op = L.op;
        P.ph[li].probs = L.probs;
        launch_coefs(L, st, coeffs, per_step, &P.ph[li].alpha, &P.ph[li].beta, &P.ph[li].beta2);
      }
      P.tall = st.kind == K_TALL;
      P.final_epi = fused ? fin.epi : EPI_F16;
      for (int t = 0; t < 3; ++t) { P.units[t] = st.prog_units[t]; P.upp[t] = st.prog_upp[t]; }
      P.recs = plan.d_recs;
      P.rec_base = bp.rec0;
      P.count = count;
      // matrices per group: the group's buffers within the L2 budget, but enough units per product to fill the grid
      // three times (a product of a group that is one wave long stalls on its predecessor's tail).  Measured on
      // config 4 (profiles/r2_program.md): groups of 2 matrices for the 4096-row buckets; 1 stalls, 3 and more spill
      // the L2 and cost clock under the power cap; the whole bucket as one group is 25 % slower than separate launches.
      const int workers = plan.sm_count / 2;
      const int fit = static_cast<int>(std::max<size_t>(1, opt.l2_group_bytes / st.mat_bytes));
      const int min_upp = std::max(1, std::min(st.prog_upp[1], st.prog_upp[2]));
      P.group = std::min(count, std::max(fit, (3 * workers + min_upp - 1) / min_upp));
      P.m_blocks = st.m_pad / kBlk;
      P.n_blocks = st.n_pad / kBlk;
      P.done = st.d_done;
      P.lr = fin.lr;
      P.lrwd = fin.lrwd;
      P.store_c = fused ? fin.store_c : true;
      P.grid = plan.sm_count;
      const bool tall = st.kind == K_TALL;
      const std::string name = std::string(!fused ? "ns_program" : fin.epi == EPI_BF16 ? "ns_program_out" : "ns_program_apply") + "[" +
                               std::to_string(tall ? st.n_pad : st.m_pad) + "x" + std::to_string(tall ? st.m_pad : st.n_pad) + "]";
      ProfScope ps(name.c_str(), stream);
      return launch_ns_program(P, stream);
    }
    for (size_t li = 0; li < nl; ++li) {
      const NsLaunch& L = it->second.launches[li];
      float alpha, beta, beta2;
      launch_coefs(L, st, coeffs, per_step, &alpha, &beta, &beta2);
      const bool last = fused && li + 1 == nl;
      std::string name = L.name;
      if (last) name.replace(name.find("_update"), 7, fin.epi == EPI_BF16 ? "_out" : "_apply");
      ProfScope ps(name.c_str(), stream);
      int rc = shape_launch(plan, st, count, bp.rec0, L.op, L.probs, alpha, beta, beta2, last ? fin : FinalEpilogue(), stream);
      if (rc) return rc;
    }
  } else {
    for (int s = 0; s < steps; ++s) {
      const float* q = coeffs + (per_step ? 3 * s : 0);
      const float a = q[0], bb = q[1], c = q[2];
      const int parity = s & 1;                 // step 0 reads Q (parity 0) and writes P
      for (int k = 0; k < count; ++k) {
        uint8_t* slot = plan.ws + st.base + static_cast<size_t>(k) * st.mat_bytes;
        float* X[2] = {reinterpret_cast<float*>(slot + st.off_q), reinterpret_cast<float*>(slot + st.off_p)};
        float* A = reinterpret_cast<float*>(slot + st.off_sq[0]);
        float* B = reinterpret_cast<float*>(slot + st.off_sq[1]);
        int rc;
        if ((rc = launch_check_gemm(OP_SYRK, X[parity], nullptr, A, st.m_pad, st.n_pad, 1.f, 0.f, stream))) return rc;
        if ((rc = launch_check_gemm(OP_SQ, A, nullptr, B, st.m_pad, st.m_pad, c, bb, stream))) return rc;
        if ((rc = launch_check_gemm(OP_BX, B, X[parity], X[1 - parity], st.m_pad, st.n_pad, 1.f, a, stream))) return rc;
      }
    }
  }
  return DMUON_OK;
}

}  // namespace dmuon
