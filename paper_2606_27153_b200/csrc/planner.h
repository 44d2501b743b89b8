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
  int force_variant[3] = {-1, -1, -1};   // per tiling op (SYRK, SQ, BX): -1 = tuned, else this tile configuration
  bool overlap = false;         // run the elementwise passes of one bucket under the GEMMs of another (side stream);
                                // measured <= 1 % on config 4 (the step is power-bound: hiding a pass saves no energy)
  bool gram_blocks = true;      // schedule "auto": Gram blocks (Eq. 4) on wide buckets; false = plain X iteration
};

struct MatrixInfo {
  int rows, cols;        // stored
  int m, n;              // oriented (m <= n)
  int m_pad, n_pad;      // padded to multiples of 128
  bool transposed;
  int bucket;
  size_t off_p, off_q;   // byte offsets into the workspace: the two m_pad x n_pad X buffers
  size_t off_sq[5];      // m_pad x m_pad buffers: G, B, and (Gram-block buckets only) B', T, R
  bool gram;             // bucket eligible for Gram blocks (wide enough that they save work)
};

// Tile configuration of one op of one bucket ("variant" of dmuon_ns_gemm).
struct TileConfig {
  bool pair = false;     // CTA-pair tiling: 256 x 256 units on two SMs (cta_group::2)
  bool quad = false;     // CTA-quad tiling: two pair units per cluster of 4, shared operand panel multicast by TMA
  int width = 2;         // single-CTA tiling, blocks per work unit: 2 -> UMMA N = 256, 1 -> N = 128
  int order = 0;         // 0: panel-major (all block rows of one column panel first), 1: row-major
};
// Variants 0..3: single CTA, (width, order) = (2,0), (1,0), (2,1), (1,1); 4, 5: CTA pair, order 0, 1.
// 6: CTA quad.  The symmetric ops have one ordering: their variants are 0, 1 (single CTA), 4 (pair) and 6 (quad).
constexpr int kNumVariants = 7;
bool variant_valid(GemmOp op, int variant);
TileConfig variant_config(int variant);

// How the k NS steps of a bucket are executed: a list of blocks whose lengths sum to k.  A block of length 1 is the
// plain step X <- (a I + B) X.  A block of length L > 1 forms G once from X, advances it in the m x m Gram space
// (G_{i+1} = P_i G_i P_i, Eq. 4), accumulates Q = P_{s+L-1} ... P_s and touches X once: X <- Q X.
// Blocks are restarts: G is always recomputed from X at the start of a block, which is what keeps fp16 storage stable
// (DESIGN.md section 6).
typedef std::vector<int> Partition;
Partition choose_partition(int steps, const float* coeffs, bool per_step, bool gram);
bool gram_eligible(int m_pad, int n_pad, bool fp32);

// How a launch's (alpha, beta, beta2) follow from the per-step coefficients (a_i, b_i, c_i).
enum CoefKind : int {
  CK_ONE = 0,    // alpha = 1                                            SYRK: G = X X^T
  CK_POLY,       // alpha = c_s1, beta = b_s1                            B = b G + c G G
  CK_A,          // alpha = 1, beta = a_s1                               T = a G + B G ; G' = a T + T B
  CK_RACC,       // alpha = 1, beta = prod a_[s0, s1), beta2 = a_s1      R' = (prod a) B' + a R + B' R
  CK_APOW        // alpha = 1, beta = prod a_[s0, s1]                    X' = (prod a) X + R X
};
struct NsLaunch {
  GemmOp op;
  CoefKind ck;
  int s0, s1;                  // step indices the coefficients come from
  GemmProblem* probs;          // device, one per matrix of the bucket
  int k_blocks, n_blocks;
  std::string name;            // profiling name: family[m_pad x n_pad]
};
struct NsProgram {
  std::vector<NsLaunch> launches;
  int x_updates = 0;           // how many times X switched buffers (result parity)
};

struct BucketPlan {
  int m_pad = 0, n_pad = 0;
  bool gram = false;
  std::vector<int> mats;               // matrix indices
  std::map<std::string, NsProgram> programs;   // by partition signature, e.g. "32"
  TileUnit* units[3] = {nullptr, nullptr, nullptr};   // per tiling op (SYRK, SQ / SQ2, BX)
  int units_per_problem[3] = {0, 0, 0};
  int variant[3] = {0, 0, 0};
  // scratch problem tables for the autotuner
  GemmProblem* tune_probs[3] = {nullptr, nullptr, nullptr};
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
  float* d_inv_norm = nullptr;
  ElemTables tables{};                 // all matrices
  std::vector<int> order;              // execution order of the buckets (most NS work first)
  std::vector<ElemTables> parts;       // per bucket, in execution order (empty: one bucket or check mode)
  cudaStream_t side = nullptr;         // side stream for the elementwise passes hidden under GEMMs
  std::vector<cudaEvent_t> ev;         // fork / join events of the overlapped step
  std::string bound_key;               // schedule signature rec.O was last bound for
  std::vector<void*> d_allocs;         // everything to cudaFree
  int sm_count = 148;
  ~Plan();
};

size_t plan_workspace_bytes(const int32_t* shapes, int count, bool fp32);
// Builds (or fetches) the plan for a shape set.  ext_ws/ext_bytes: caller workspace or (nullptr, 0).
int get_plan(const int32_t* shapes, int count, const Options& opt, void* ext_ws, size_t ext_bytes, cudaStream_t stream,
             Plan** out);
void drop_plans();

// Enqueue k NS steps over every bucket of the plan; X0 is in buffer Q.  result_parity(...) tells where a bucket's
// result ends (0 = Q, 1 = P) for the same arguments.
int run_ns_steps(Plan& plan, int steps, const float* coeffs, bool per_step, const Options& opt, cudaStream_t stream);
int run_ns_bucket(Plan& plan, int bucket, int steps, const float* coeffs, bool per_step, const Options& opt,
                  cudaStream_t stream);
int result_parity(const Plan& plan, const BucketPlan& b, int steps, const float* coeffs, bool per_step, const Options& opt);
std::string partition_key(const Partition& p);

// Build tile units for an op.
std::vector<TileUnit> make_units(GemmOp op, int m_blocks, int n_blocks, const TileConfig& cfg);
int encode_tmap_2d(CUtensorMap* out, const void* base, uint64_t rows, uint64_t cols, uint32_t box_cols,
                   uint32_t box_rows);
int fill_problem(GemmProblem& g, GemmOp op, const void* a_mat, uint64_t a_rows, uint64_t a_cols, const void* b_mat,
                 uint64_t b_rows, uint64_t b_cols, const void* d, void* c, int ldc, const void* d2 = nullptr);
int check_device();

}  // namespace dmuon
