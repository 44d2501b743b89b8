// Host-side planner: buckets, workspace layout, TMA descriptors, grouped-launch tables, autotune + persistent cache.
// See planner.h.  (PAPER.md:180 batching by shape; PAPER.md:184 autotuner and persistent kernel cache.)
#include "planner.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <fstream>
#include <sstream>
#include <sys/stat.h>

namespace dmuon {

// Gram blocks replace 2 (L - 1) of the m x n products of L steps by 4 (L - 1) m x m products: worth it when the matrix
// is wide.  Tiny Gram matrices (one block) stay on the plain iteration (latency-bound either way).
bool gram_eligible(int m_pad, int n_pad, bool fp32) { return !fp32 && m_pad >= 2 * kBlk && 2 * n_pad >= 3 * m_pad; }

namespace {

std::vector<std::unique_ptr<Plan>> g_plans;
std::map<std::string, int> g_tune_cache;     // "op m_pad n_pad count" -> variant
bool g_tune_loaded = false;
std::string g_tune_loaded_path;

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
inline int pad128(int v) { return (v + kBlk - 1) / kBlk * kBlk; }

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

void describe(const int32_t* shapes, int count, std::vector<MatrixInfo>& mats, size_t es, size_t* ws_bytes) {
  mats.resize(count);
  size_t off = 0;
  for (int i = 0; i < count; ++i) {
    MatrixInfo& mi = mats[i];
    mi.rows = shapes[2 * i];
    mi.cols = shapes[2 * i + 1];
    mi.transposed = mi.rows > mi.cols;            // work in the smaller Gram dimension
    mi.m = std::min(mi.rows, mi.cols);
    mi.n = std::max(mi.rows, mi.cols);
    mi.m_pad = pad128(mi.m);
    mi.n_pad = pad128(mi.n);
    mi.bucket = -1;
    const size_t xb = align_up(static_cast<size_t>(mi.m_pad) * mi.n_pad * es, 1024);
    const size_t ab = align_up(static_cast<size_t>(mi.m_pad) * mi.m_pad * es, 1024);
    mi.gram = gram_eligible(mi.m_pad, mi.n_pad, es == 4);
    mi.off_p = off; off += xb;
    mi.off_q = off; off += xb;
    for (int k = 0; k < 5; ++k) {
      mi.off_sq[k] = off;
      if (k < 2 || mi.gram) off += ab;
    }
  }
  *ws_bytes = off;
}

std::string resolve_cache_path(const Options& opt) {
  if (opt.cache_path_set) return opt.cache_path;
  if (const char* e = getenv("DMUON_CACHE")) return e;
  if (const char* h = getenv("HOME")) return std::string(h) + "/.cache/dmuon/tune.txt";
  return "";
}

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
    std::string tag;
    int op, m, n, cnt, variant;
    if (ss >> tag >> op >> m >> n >> cnt >> variant && tag == "v4" && variant >= 0 && variant < kNumVariants) {
      char key[96];
      snprintf(key, sizeof key, "%d %d %d %d", op, m, n, cnt);
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
  for (auto& kv : g_tune_cache) out << "v4 " << kv.first << " " << kv.second << "\n";
}

inline int tiling_op(GemmOp op) { return op == OP_SQ2 ? OP_SQ : op; }   // SQ2 shares SQ's units and variant

int bucket_launch(const Plan& plan, const BucketPlan& b, GemmOp op, const GemmProblem* probs, float alpha, float beta,
                  float beta2, cudaStream_t stream, const TileUnit* units_override = nullptr, int upp_override = 0,
                  int variant_override = -1) {
  const int top = tiling_op(op);
  const bool pair = variant_config(variant_override >= 0 ? variant_override : b.variant[top]).pair;
  GemmLaunch L;
  L.op = op;
  L.problems = probs;
  L.units = units_override ? units_override : b.units[top];
  L.units_per_problem = units_override ? upp_override : b.units_per_problem[top];
  L.num_problems = static_cast<int>(b.mats.size());
  L.k_blocks = (op == OP_SYRK ? b.n_pad : b.m_pad) / kBlkK;
  L.m_blocks = b.m_pad / kBlk;
  L.n_blocks = (op == OP_BX ? b.n_pad : b.m_pad) / kBlk;
  L.pair = pair;
  L.quad = variant_config(variant_override >= 0 ? variant_override : b.variant[top]).quad;
  L.alpha = alpha;
  L.beta = beta;
  L.beta2 = beta2;
  L.grid = plan.sm_count;
  return launch_ns_gemm(L, stream);
}

// Time each variant of each op of a bucket on the plan's own (scratch) workspace and keep the fastest.
int autotune_bucket(Plan& plan, BucketPlan& b, const Options& opt, cudaStream_t stream) {
  const std::string path = resolve_cache_path(opt);
  load_tune_cache(path);
  bool dirty = false;
  for (int op = 0; op < 3; ++op) {
    char key[96];
    snprintf(key, sizeof key, "%d %d %d %d", op, b.m_pad, b.n_pad, static_cast<int>(b.mats.size()));
    auto it = g_tune_cache.find(key);
    int best = 0;
    if (opt.force_variant[op] >= 0 && variant_valid(static_cast<GemmOp>(op), opt.force_variant[op])) {
      best = opt.force_variant[op];
    } else if (it != g_tune_cache.end()) {
      best = it->second;
    } else if (opt.autotune) {
      cudaEvent_t e0, e1;
      DMUON_CUDA_CHECK(cudaEventCreate(&e0));
      DMUON_CUDA_CHECK(cudaEventCreate(&e1));
      // the CTA-pair tilings are the incumbents: another configuration has to beat them by 10 % in this short, isolated
      // measurement to be taken.  Timer noise must not flip the choice between runs, and a few launches at boost clock
      // flatter the single-CTA tilings: they move 1.5x the L2->SMEM bytes per FLOP, which costs them more once the
      // board sits at its power cap (measured: 25.8 against 18.4 ms per step for B = bG + cGG on 64 x 4096^2).  Unit order of the X update: row-major while X stays in
      // L2, column-panel-major beyond (row-major then streams the whole X once per block row: measured 16 GB instead
      // of 2.7 GB of DRAM reads per 12 matrices of 4096 x 14336)
      const bool x_in_l2 = static_cast<size_t>(b.m_pad) * b.n_pad * sizeof(__half) <= (48u << 20);
      const int preferred = op == OP_BX ? (x_in_l2 ? 5 : 4) : 4;
      float best_ms = 1e30f, preferred_ms = 1e30f;
      for (int v = 0; v < kNumVariants; ++v) {
        if (!variant_valid(static_cast<GemmOp>(op), v)) continue;
        const TileConfig cfg = variant_config(v);
        // The quad tiling measured slower than the pair tiling on every bucket tried (TMA multicast at cluster size 4
        // saves no L2 traffic over concurrent unicast loads, and only 33 clusters of 4 are co-resident on 148 SMs): it
        // stays available through option "variants" but is not a tuning candidate.
        if (cfg.quad) continue;
        std::vector<TileUnit> hu = make_units(static_cast<GemmOp>(op), b.m_pad / kBlk, b.n_pad / kBlk, cfg);
        TileUnit* du = nullptr;
        DMUON_CUDA_CHECK(cudaMalloc(&du, hu.size() * sizeof(TileUnit)));
        DMUON_CUDA_CHECK(cudaMemcpy(du, hu.data(), hu.size() * sizeof(TileUnit), cudaMemcpyHostToDevice));
        int rc = DMUON_OK;
        float ms = 1e30f;
        for (int rep = 0; rep < 4 && rc == DMUON_OK; ++rep) {   // rep 0 warms up
          cudaEventRecord(e0, stream);
          rc = bucket_launch(plan, b, static_cast<GemmOp>(op), b.tune_probs[op], 1.f, 0.f, 0.f, stream, du, static_cast<int>(hu.size()), v);
          cudaEventRecord(e1, stream);
          if (cudaEventSynchronize(e1) != cudaSuccess) rc = DMUON_ERR_CUDA;
          float t = 0.f;
          cudaEventElapsedTime(&t, e0, e1);
          if (rep > 0) ms = std::min(ms, t);
        }
        cudaFree(du);
        if (rc) { cudaEventDestroy(e0); cudaEventDestroy(e1); set_error("autotune launch failed"); return rc; }
        if (ms < best_ms) { best_ms = ms; best = v; }
        if (v == preferred) preferred_ms = ms;
      }
      if (best != preferred && best_ms > 0.90f * preferred_ms) best = preferred;
      cudaEventDestroy(e0);
      cudaEventDestroy(e1);
      g_tune_cache[key] = best;
      dirty = true;
    }
    b.variant[op] = best;
  }
  if (dirty) save_tune_cache(path);
  return DMUON_OK;
}

}  // namespace

int fill_problem(GemmProblem& g, GemmOp op, const void* a_mat, uint64_t a_rows, uint64_t a_cols, const void* b_mat,
                 uint64_t b_rows, uint64_t b_cols, const void* d, void* c, int ldc, const void* d2) {
  memset(&g, 0, sizeof g);
  int rc = encode_tmap_2d(&g.tmA, a_mat, a_rows, a_cols, kBlkK, kBlk);
  if (rc) return rc;
  if (op == OP_BX) rc = encode_tmap_2d(&g.tmB, b_mat, b_rows, b_cols, 64, kBlkK);   // MN-major: 64 (n) x 64 (k) boxes
  else rc = encode_tmap_2d(&g.tmB, b_mat, b_rows, b_cols, kBlkK, kBlk);
  if (rc) return rc;
  g.D = static_cast<const __half*>(d);
  g.C = static_cast<__half*>(c);
  g.D2 = static_cast<const __half*>(d2);
  g.ldc = ldc;
  return DMUON_OK;
}

Plan::~Plan() {
  for (void* p : d_allocs) cudaFree(p);
  for (cudaEvent_t e : ev) cudaEventDestroy(e);
  if (side) cudaStreamDestroy(side);
}

TileConfig variant_config(int variant) {
  TileConfig c;
  if (variant == 6) {
    c.pair = true;
    c.quad = true;
    c.order = 1;
    return c;
  }
  if (variant >= 4) {
    c.pair = true;
    c.order = variant & 1;
  } else {
    c.width = (variant & 1) ? 1 : 2;
    c.order = (variant >> 1) & 1;
  }
  return c;
}

bool variant_valid(GemmOp op, int variant) {
  if (variant < 0 || variant >= kNumVariants) return false;
  if (variant == 6) return true;
  return op == OP_BX || variant_config(variant).order == 0;   // symmetric ops have one ordering
}

std::vector<TileUnit> make_units(GemmOp op, int mb, int nb, const TileConfig& cfg) {
  std::vector<TileUnit> u;
  auto push = [&](int i, int j, int w) { u.push_back(TileUnit{static_cast<int16_t>(i), static_cast<int16_t>(j), static_cast<int16_t>(w), 0}); };
  if (cfg.quad) {
    // two 256 x 256 units per entry, sharing a block row (pairs along a row) or a block column (leftovers of rows
    // with an odd number of units, paired down the last column); a final odd unit is paired with itself
    const int MB = (mb + 1) / 2, NB = (nb + 1) / 2;
    auto quad = [&](int m0, int n0, int m1, int n1) {
      u.push_back(TileUnit{static_cast<int16_t>(m0), static_cast<int16_t>(n0), static_cast<int16_t>(m1), static_cast<int16_t>(n1)});
    };
    const int ncols = op == OP_BX ? NB : MB;
    std::vector<std::pair<int, int>> left;
    for (int i = 0; i < MB; ++i) {
      int j = op == OP_BX ? 0 : i;
      for (; j + 1 < ncols; j += 2) quad(i, j, i, j + 1);
      if (j < ncols) left.push_back({i, j});
    }
    for (size_t k = 0; k + 1 < left.size(); k += 2) quad(left[k].first, left[k].second, left[k + 1].first, left[k + 1].second);
    if (left.size() % 2) quad(left.back().first, left.back().second, left.back().first, left.back().second);
    return u;
  }
  if (cfg.pair) {
    // 256 x 256 units; an odd block count leaves a half-empty last unit (operands zero-filled, stores skipped)
    const int MB = (mb + 1) / 2, NB = (nb + 1) / 2;
    if (op == OP_BX) {
      if (cfg.order == 0) { for (int j = 0; j < NB; ++j) for (int i = 0; i < MB; ++i) push(i, j, 2); }
      else                { for (int i = 0; i < MB; ++i) for (int j = 0; j < NB; ++j) push(i, j, 2); }
    } else {
      for (int i = 0; i < MB; ++i) for (int j = i; j < MB; ++j) push(i, j, 2);
    }
    return u;
  }
  if (op == OP_BX) {
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
                   uint32_t box_rows) {
  int rc = load_encode();
  if (rc) return rc;
  const cuuint64_t gdim[2] = {cols, rows};
  const cuuint64_t gstride[1] = {cols * sizeof(__half)};
  const cuuint32_t box[2] = {box_cols, box_rows};
  const cuuint32_t estr[2] = {1, 1};
  CUresult r = g_encode(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, const_cast<void*>(base), gdim, gstride, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    set_error("cuTensorMapEncodeTiled failed (%d) for %llu x %llu, box %u x %u, base %p", static_cast<int>(r),
              static_cast<unsigned long long>(rows), static_cast<unsigned long long>(cols), box_rows, box_cols, base);
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
  return DMUON_OK;
}

size_t plan_workspace_bytes(const int32_t* shapes, int count, bool fp32) {
  std::vector<MatrixInfo> mats;
  size_t bytes = 0;
  describe(shapes, count, mats, fp32 ? 4 : 2, &bytes);
  return bytes;
}

void drop_plans() { g_plans.clear(); }

int get_plan(const int32_t* shapes, int count, const Options& opt, void* ext_ws, size_t ext_bytes, cudaStream_t stream,
             Plan** out) {
  for (auto& up : g_plans) {
    Plan& p = *up;
    if (p.fp32 == opt.fp32_check && p.shapes.size() == static_cast<size_t>(2 * count) &&
        (count == 0 || memcmp(p.shapes.data(), shapes, sizeof(int32_t) * 2 * count) == 0)) {
      *out = &p;
      return DMUON_OK;
    }
  }
  int rc = check_device();
  if (rc) return rc;

  std::unique_ptr<Plan> up(new Plan);
  Plan& p = *up;
  p.shapes.assign(shapes, shapes + 2 * count);
  p.fp32 = opt.fp32_check;
  const size_t es = p.fp32 ? 4 : 2;
  describe(shapes, count, p.mats, es, &p.ws_bytes);
  int dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&p.sm_count, cudaDevAttrMultiProcessorCount, dev);

  // ---- workspace
  if (ext_ws) {
    if (ext_bytes < p.ws_bytes) {
      set_error("caller workspace of %zu bytes is smaller than the %zu bytes this shape set needs", ext_bytes, p.ws_bytes);
      return DMUON_ERR_OOM;
    }
    p.ws = static_cast<uint8_t*>(ext_ws);
  } else {
    rc = dev_alloc(p, &p.ws, p.ws_bytes);
    if (rc) return rc;
    p.ws_owned = true;
  }

  // scratch contents for the autotuner (tensor-core mode) / zeros (check mode)
  if (!p.fp32) { if ((rc = launch_fill_scratch(p.ws, p.ws_bytes, stream))) return rc; }
  else DMUON_CUDA_CHECK(cudaMemsetAsync(p.ws, 0, p.ws_bytes, stream));

  // ---- buckets by padded oriented shape
  std::map<std::pair<int, int>, int> bucket_of;
  for (int i = 0; i < count; ++i) {
    MatrixInfo& mi = p.mats[i];
    auto key = std::make_pair(mi.m_pad, mi.n_pad);
    auto it = bucket_of.find(key);
    if (it == bucket_of.end()) {
      it = bucket_of.emplace(key, static_cast<int>(p.buckets.size())).first;
      p.buckets.emplace_back();
      p.buckets.back().m_pad = mi.m_pad;
      p.buckets.back().n_pad = mi.n_pad;
    }
    mi.bucket = it->second;
    p.buckets[it->second].mats.push_back(i);
  }

  // ---- elementwise tables.  One set over all matrices (`tables`) and, when there are several buckets, one set per
  //      bucket (`parts`, in execution order) in which the matrices of the other buckets have no work items: the step
  //      runs the elementwise passes of one bucket on a side stream under the GEMMs of another (api.cu).
  p.h_recs.resize(count);
  for (int i = 0; i < count; ++i) {
    const MatrixInfo& mi = p.mats[i];
    MatRec& r = p.h_recs[i];
    memset(&r, 0, sizeof r);
    r.U = p.ws + mi.off_p;
    r.X0 = p.ws + mi.off_q;
    r.O = nullptr;
    r.rows = mi.rows; r.cols = mi.cols;
    r.m_pad = mi.m_pad; r.n_pad = mi.n_pad;
    r.transposed = mi.transposed ? 1 : 0;
    r.scale = static_cast<float>(std::sqrt(std::max(1.0, static_cast<double>(mi.rows) / mi.cols)));   // reading N4
  }
  if ((rc = dev_alloc(p, &p.d_recs, count))) return rc;
  if ((rc = dev_alloc(p, &p.d_inv_norm, count))) return rc;
  auto build_tables = [&](int only_bucket, ElemTables* out) -> int {
    std::vector<int64_t> flat_prefix(count + 1, 0), tile_prefix(count + 1, 0), ptile_prefix(count + 1, 0);
    std::vector<int64_t> fa_prefix(count + 1, 0), fb_prefix(count + 1, 0);
    for (int i = 0; i < count; ++i) {
      const MatrixInfo& mi = p.mats[i];
      const bool member = only_bucket < 0 || mi.bucket == only_bucket;
      const int64_t elems = static_cast<int64_t>(mi.rows) * mi.cols;
      // normalise / apply path of this matrix: A (flat), B (16-bit tile transpose) or the generic tiles
      const bool aligned = !p.fp32 && mi.rows % kBlk == 0 && mi.cols % kBlk == 0;
      const bool path_a = aligned && !mi.transposed, path_b = aligned && mi.transposed;
      const bool generic = !path_a && !path_b;
      flat_prefix[i + 1] = flat_prefix[i] + (member ? (elems + kFlatChunk - 1) / kFlatChunk : 0);
      fa_prefix[i + 1] = fa_prefix[i] + (member && path_a ? elems / kFlatChunk : 0);
      fb_prefix[i + 1] = fb_prefix[i] + (member && path_b ? static_cast<int64_t>(mi.rows / kTile) * (mi.cols / kTile) : 0);
      tile_prefix[i + 1] = tile_prefix[i] + (member && generic ? static_cast<int64_t>((mi.rows + kTile - 1) / kTile) * ((mi.cols + kTile - 1) / kTile) : 0);
      ptile_prefix[i + 1] = ptile_prefix[i] + (member && generic ? static_cast<int64_t>(mi.m_pad / kTile) * (mi.n_pad / kTile) : 0);
    }
    int64_t *d_flat = nullptr, *d_tile = nullptr, *d_ptile = nullptr, *d_fa = nullptr, *d_fb = nullptr;
    float* d_partials = nullptr;
    int r2;
    if ((r2 = upload(p, &d_flat, flat_prefix))) return r2;
    if ((r2 = upload(p, &d_tile, tile_prefix))) return r2;
    if ((r2 = upload(p, &d_ptile, ptile_prefix))) return r2;
    if ((r2 = upload(p, &d_fa, fa_prefix))) return r2;
    if ((r2 = upload(p, &d_fb, fb_prefix))) return r2;
    if ((r2 = dev_alloc(p, &d_partials, static_cast<size_t>(flat_prefix[count])))) return r2;
    out->recs = p.d_recs;
    out->flat_prefix = d_flat;
    out->tile_prefix = d_tile;
    out->ptile_prefix = d_ptile;
    out->fa_prefix = d_fa;
    out->fb_prefix = d_fb;
    out->count = count;
    out->flat_chunks = flat_prefix[count];
    out->tiles = tile_prefix[count];
    out->ptiles = ptile_prefix[count];
    out->fa_chunks = fa_prefix[count];
    out->fb_tiles = fb_prefix[count];
    out->partials = d_partials;
    out->inv_norm = p.d_inv_norm;
    return DMUON_OK;
  };
  if ((rc = build_tables(-1, &p.tables))) return rc;
  // execution order of the buckets: most NS work first, so that the largest elementwise passes that can be hidden
  // (normalise of the later buckets, apply of the earlier ones) run under the longest GEMM phases
  p.order.resize(p.buckets.size());
  for (size_t b = 0; b < p.buckets.size(); ++b) p.order[b] = static_cast<int>(b);
  auto cost = [&](int b) {
    const BucketPlan& bp = p.buckets[b];
    return static_cast<double>(bp.mats.size()) * bp.m_pad * bp.m_pad * (2.0 * bp.n_pad + bp.m_pad);
  };
  std::stable_sort(p.order.begin(), p.order.end(), [&](int a, int b) { return cost(a) > cost(b); });
  if (!p.fp32 && p.buckets.size() > 1) {
    p.parts.resize(p.buckets.size());
    for (size_t k = 0; k < p.order.size(); ++k)
      if ((rc = build_tables(p.order[k], &p.parts[k]))) return rc;
    DMUON_CUDA_CHECK(cudaStreamCreateWithFlags(&p.side, cudaStreamNonBlocking));
    p.ev.resize(2 * p.buckets.size() + 2);
    for (cudaEvent_t& e : p.ev) DMUON_CUDA_CHECK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
  }

  // ---- grouped GEMM tables (tensor-core mode only): scratch problems for the autotuner, tile units per op.  The
  //      launch programs of the NS steps are built on first use (build_program), they depend on the step count.
  if (!p.fp32) {
    for (BucketPlan& b : p.buckets) {
      const size_t nprob = b.mats.size();
      b.gram = p.mats[b.mats[0]].gram;
      std::vector<GemmProblem> tp[3];
      for (int op = 0; op < 3; ++op) tp[op].resize(nprob);
      for (size_t k = 0; k < nprob; ++k) {
        const MatrixInfo& mi = p.mats[b.mats[k]];
        void* XQ = p.ws + mi.off_q;
        void* XP = p.ws + mi.off_p;
        void* A = p.ws + mi.off_sq[0];
        void* B = p.ws + mi.off_sq[1];
        const uint64_t m = mi.m_pad, n = mi.n_pad;
        if ((rc = fill_problem(tp[OP_SYRK][k], OP_SYRK, XQ, m, n, XQ, m, n, nullptr, A, mi.m_pad))) return rc;
        if ((rc = fill_problem(tp[OP_SQ][k], OP_SQ, A, m, m, A, m, m, A, B, mi.m_pad))) return rc;
        if ((rc = fill_problem(tp[OP_BX][k], OP_BX, B, m, m, XQ, m, n, XQ, XP, mi.n_pad))) return rc;
      }
      for (int op = 0; op < 3; ++op)
        if ((rc = upload(p, &b.tune_probs[op], tp[op]))) return rc;
      // tile configuration: tuned (cache or measurement) or default variant 0
      if ((rc = autotune_bucket(p, b, opt, stream))) return rc;
      for (int op = 0; op < 3; ++op) {
        std::vector<TileUnit> hu = make_units(static_cast<GemmOp>(op), b.m_pad / kBlk, b.n_pad / kBlk, variant_config(b.variant[op]));
        b.units_per_problem[op] = static_cast<int>(hu.size());
        if ((rc = upload(p, &b.units[op], hu))) return rc;
      }
    }
  }
  DMUON_CUDA_CHECK(cudaDeviceSynchronize());
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

int result_parity(const Plan& plan, const BucketPlan& b, int steps, const float* coeffs, bool per_step, const Options& opt) {
  if (plan.fp32) return steps & 1;
  return static_cast<int>(choose_partition(steps, coeffs, per_step, b.gram && opt.gram_blocks).size()) & 1;
}

namespace {

// Build the launch list of one bucket for a partition of the steps into blocks.  m x m buffers: 0 = G, 1/2 = B and B'
// (alternating), 3 = T, 4 = R.
int build_program(Plan& p, BucketPlan& b, const Partition& part, NsProgram& prog) {
  const size_t nprob = b.mats.size();
  const int kb_n = b.n_pad / kBlkK, kb_m = b.m_pad / kBlkK, nb_m = b.m_pad / kBlk, nb_n = b.n_pad / kBlk;
  int rc;
  auto emit = [&](GemmOp op, CoefKind ck, int s0, int s1, const char* name, int a_buf, int b_buf, int d_buf, int d2_buf,
                  int c_buf, int xsrc) -> int {
    // buffer ids: 0..4 = m x m buffers; 10 / 11 = X in Q / P
    std::vector<GemmProblem> hp(nprob);
    for (size_t k = 0; k < nprob; ++k) {
      const MatrixInfo& mi = p.mats[b.mats[k]];
      auto buf = [&](int id) -> void* {
        if (id < 0) return nullptr;
        if (id >= 10) return p.ws + (id == 10 ? mi.off_q : mi.off_p);
        return p.ws + mi.off_sq[id];
      };
      const uint64_t m = mi.m_pad, n = mi.n_pad;
      if (op == OP_SYRK) rc = fill_problem(hp[k], op, buf(xsrc), m, n, buf(xsrc), m, n, nullptr, buf(c_buf), mi.m_pad);
      else if (op == OP_BX) rc = fill_problem(hp[k], op, buf(a_buf), m, m, buf(xsrc), m, n, buf(xsrc), buf(c_buf), mi.n_pad);
      else rc = fill_problem(hp[k], op, buf(a_buf), m, m, buf(b_buf), m, m, buf(d_buf), buf(c_buf), mi.m_pad, buf(d2_buf));
      if (rc) return rc;
    }
    NsLaunch L;
    L.op = op; L.ck = ck; L.s0 = s0; L.s1 = s1;
    L.name = std::string(name) + "[" + std::to_string(b.m_pad) + "x" + std::to_string(b.n_pad) + "]";
    L.k_blocks = op == OP_SYRK ? kb_n : kb_m;
    L.n_blocks = op == OP_BX ? nb_n : nb_m;
    if ((rc = upload(p, &L.probs, hp))) return rc;
    prog.launches.push_back(L);
    return DMUON_OK;
  };
  int s = 0, par = 0;   // X0 is in Q (parity 0)
  for (int L : part) {
    if (L > 1 && !b.gram) { set_error("internal: Gram block on a bucket without Gram buffers"); return DMUON_ERR_INVALID_ARG; }
    if (L > 3) { set_error("internal: Gram block longer than 3"); return DMUON_ERR_INVALID_ARG; }
    const int xs = 10 + par, xd = 10 + (1 - par);
    int g = 0, bc = 1, bn = 2, t = 3, r = 1;     // R_0 = B_0 (alias)
    if ((rc = emit(OP_SYRK, CK_ONE, s, s, "ns_syrk_xxt", -1, -1, -1, -1, g, xs))) return rc;            // G = X X^T
    if ((rc = emit(OP_SQ, CK_POLY, s, s, "ns_sq_poly", g, g, g, -1, bc, -1))) return rc;                // B = b G + c G G
    for (int i = 1; i < L; ++i) {
      const int st = s + i;
      if ((rc = emit(OP_SQ, CK_A, st - 1, st - 1, "ns_gram_mm", bc, g, g, -1, t, -1))) return rc;       // T = a G + B G
      if ((rc = emit(OP_SQ, CK_A, st - 1, st - 1, "ns_gram_mm", t, bc, t, -1, g, -1))) return rc;       // G' = a T + T B
      if ((rc = emit(OP_SQ, CK_POLY, st, st, "ns_sq_poly", g, g, g, -1, bn, -1))) return rc;            // B' = b G' + c G' G'
      const int rn = (i == 1) ? 4 : t;            // free buffer: R (i = 1), then T (not needed after G')
      if ((rc = emit(OP_SQ2, CK_RACC, s, st, "ns_gram_mm", bn, r, bn, r, rn, -1))) return rc;            // R' = (prod a) B' + a R + B' R
      r = rn;
      const int tmp = bc; bc = bn; bn = tmp;
    }
    if ((rc = emit(OP_BX, CK_APOW, s, s + L - 1, "ns_bx_update", r, -1, -1, -1, xd, xs))) return rc;     // X' = (prod a) X + R X
    s += L;
    par ^= 1;
    ++prog.x_updates;
  }
  return DMUON_OK;
}

void launch_coefs(const NsLaunch& L, const float* coeffs, bool per_step, float* alpha, float* beta, float* beta2) {
  auto co = [&](int step, int which) { return coeffs[(per_step ? 3 * step : 0) + which]; };
  *alpha = 1.f; *beta = 0.f; *beta2 = 0.f;
  double prod = 1.0;
  switch (L.ck) {
    case CK_ONE: break;
    case CK_POLY: *alpha = co(L.s1, 2); *beta = co(L.s1, 1); break;
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

int run_ns_steps(Plan& plan, int steps, const float* coeffs, bool per_step, const Options& opt, cudaStream_t stream) {
  for (int bi : plan.order) {
    int rc = run_ns_bucket(plan, bi, steps, coeffs, per_step, opt, stream);
    if (rc) return rc;
  }
  return DMUON_OK;
}

int run_ns_bucket(Plan& plan, int bucket, int steps, const float* coeffs, bool per_step, const Options& opt,
                  cudaStream_t stream) {
  {
    BucketPlan& b = plan.buckets[bucket];
    if (!plan.fp32) {
      const Partition part = choose_partition(steps, coeffs, per_step, b.gram && opt.gram_blocks);
      const std::string key = partition_key(part);
      auto it = b.programs.find(key);
      if (it == b.programs.end()) {
        NsProgram prog;
        int rc = build_program(plan, b, part, prog);
        if (rc) return rc;
        it = b.programs.emplace(key, std::move(prog)).first;
      }
      for (const NsLaunch& L : it->second.launches) {
        float alpha, beta, beta2;
        launch_coefs(L, coeffs, per_step, &alpha, &beta, &beta2);
        ProfScope ps(L.name.c_str(), stream);
        int rc = bucket_launch(plan, b, L.op, L.probs, alpha, beta, beta2, stream);
        if (rc) return rc;
      }
    } else {
      for (int s = 0; s < steps; ++s) {
        const float* q = coeffs + (per_step ? 3 * s : 0);
        const float a = q[0], bb = q[1], c = q[2];
        const int parity = s & 1;                 // step 0 reads Q (parity 0) and writes P
        for (int idx : b.mats) {
          const MatrixInfo& mi = plan.mats[idx];
          float* X[2] = {reinterpret_cast<float*>(plan.ws + mi.off_q), reinterpret_cast<float*>(plan.ws + mi.off_p)};
          float* A = reinterpret_cast<float*>(plan.ws + mi.off_sq[0]);
          float* B = reinterpret_cast<float*>(plan.ws + mi.off_sq[1]);
          int rc;
          if ((rc = launch_check_gemm(OP_SYRK, X[parity], nullptr, A, mi.m_pad, mi.n_pad, 1.f, 0.f, stream))) return rc;
          if ((rc = launch_check_gemm(OP_SQ, A, nullptr, B, mi.m_pad, mi.m_pad, c, bb, stream))) return rc;
          if ((rc = launch_check_gemm(OP_BX, B, X[parity], X[1 - parity], mi.m_pad, mi.n_pad, 1.f, a, stream))) return rc;
        }
      }
    }
  }
  return DMUON_OK;
}

}  // namespace dmuon
