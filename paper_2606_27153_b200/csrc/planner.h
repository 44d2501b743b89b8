// Host-side planner of libdmuon: groups the heterogeneous matrices of a call into shape buckets (PAPER.md:180,
// "grouped by shape and advanced ... together"), lays out the workspace, builds the TMA descriptors and grouped
// launch tables once, and picks each bucket's tile configuration by on-device measurement with a persistent
// cache keyed by problem shape and op (Fig. 6).
#pragma once

#include <map>
#include <memory>

#include "common.h"

namespace dmuon {

struct Options {
  int steps = 5;
  float coeffs[3] = {3.4445f, -4.7750f, 2.0315f};
  bool fp32_check = false;
  bool autotune = true;
  bool profile = false;
  std::string cache_path;       // resolved lazily
  bool cache_path_set = false;
  float eps = 1e-7f;
};

struct MatrixInfo {
  int rows, cols;        // stored
  int m, n;              // oriented (m <= n)
  int m_pad, n_pad;      // padded to multiples of 128
  bool transposed;
  int bucket;
  size_t off_p, off_q, off_a, off_b;   // byte offsets into the workspace
};

// Tile configuration of one op of one bucket ("variant" of dmuon_ns_gemm).
struct TileConfig {
  bool pair = false;     // CTA-pair tiling: 256 x 256 units on two SMs (cta_group::2)
  int width = 2;         // single-CTA tiling, blocks per work unit: 2 -> UMMA N = 256, 1 -> N = 128
  int order = 0;         // 0: panel-major (all block rows of one column panel first), 1: row-major
};
// Variants 0..3: single CTA, (width, order) = (2,0), (1,0), (2,1), (1,1); 4, 5: CTA pair, order 0, 1.
// The symmetric ops have one ordering: their variants are 0, 1 (single CTA) and 4 (pair).
constexpr int kNumVariants = 6;
bool variant_valid(GemmOp op, int variant);
TileConfig variant_config(int variant);

struct BucketPlan {
  int m_pad = 0, n_pad = 0;
  std::vector<int> mats;               // matrix indices
  // device tables
  GemmProblem* syrk[2] = {nullptr, nullptr};   // [src parity]: 0 = X in Q, 1 = X in P
  GemmProblem* sq = nullptr;
  GemmProblem* bx[2] = {nullptr, nullptr};     // [src parity]: 0 = Q -> P, 1 = P -> Q
  TileUnit* units[3] = {nullptr, nullptr, nullptr};   // per op
  int units_per_problem[3] = {0, 0, 0};
  int variant[3] = {0, 0, 0};
};

struct Plan {
  std::vector<int32_t> shapes;         // key
  bool fp32 = false;
  std::vector<MatrixInfo> mats;
  std::vector<BucketPlan> buckets;
  size_t ws_bytes = 0;
  uint8_t* ws = nullptr;               // device workspace (owned unless external)
  bool ws_owned = false;
  // elementwise tables
  std::vector<MatRec> h_recs;          // host mirror (pointers patched per call)
  MatRec* d_recs = nullptr;
  int64_t *d_flat_prefix = nullptr, *d_tile_prefix = nullptr, *d_ptile_prefix = nullptr;
  float *d_partials = nullptr, *d_inv_norm = nullptr;
  ElemTables tables{};
  int o_parity = -1;                   // which buffer rec.O points at (steps & 1), -1 = unset
  // staging for the _host entry point
  uint8_t* stage = nullptr;            // W | G | M device copies
  std::vector<size_t> stage_off;       // per matrix offset of W; G at +stage_third, M at +2*stage_third
  size_t stage_third = 0;
  std::vector<void*> d_allocs;         // everything to cudaFree
  int sm_count = 148;
  ~Plan();
};

size_t plan_workspace_bytes(const int32_t* shapes, int count, bool fp32);
// Builds (or fetches) the plan for a shape set.  ext_ws/ext_bytes: caller workspace or (nullptr, 0).
int get_plan(const int32_t* shapes, int count, const Options& opt, void* ext_ws, size_t ext_bytes, cudaStream_t stream,
             Plan** out);
void drop_plans();

// Enqueue k NS steps over every bucket of the plan; X0 is in buffer Q; result ends in P if steps is odd, else Q.
int run_ns_steps(Plan& plan, int steps, const float* coeffs, bool per_step, cudaStream_t stream);

// Build tile units for an op.
std::vector<TileUnit> make_units(GemmOp op, int m_blocks, int n_blocks, const TileConfig& cfg);
int encode_tmap_2d(CUtensorMap* out, const void* base, uint64_t rows, uint64_t cols, uint32_t box_cols,
                   uint32_t box_rows);
int fill_problem(GemmProblem& g, GemmOp op, const void* a_mat, uint64_t a_rows, uint64_t a_cols, const void* b_mat,
                 uint64_t b_rows, uint64_t b_cols, const void* d, void* c, int ldc);
int check_device();

}  // namespace dmuon
