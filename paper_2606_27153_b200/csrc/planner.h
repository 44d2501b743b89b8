// Host-side planner of libdmuon: groups the heterogeneous matrices of a call into shape buckets (PAPER.md:180,
// "grouped by shape and advanced ... together"), lays out ONE workspace region that the buckets use one after the
// other, builds the TMA descriptors and grouped launch tables once per bucket shape, and picks each bucket shape's
// tile configuration by on-device measurement with a persistent cache keyed by problem shape and op (PAPER.md:184,
// Fig. 6).
#pragma once

#include <map>
#include <memory>

#include "common.h"

namespace dmuon {

struct Options {
  int steps = 5;
  float coeffs[3] = {3.4445f, -4.7750f, 2.0315f};
  std::vector<float> sched;     // option "coeffs_sched": one (a, b, c) per step for the Muon-step entry points
                                // (per-step sets such as Polar Express); empty = `coeffs` at every step
  bool fp32_check = false;
  bool autotune = true;
  bool profile = false;
  std::string cache_path;       // resolved lazily
  bool cache_path_set = false;
  float eps = 1e-7f;
  int force_variant[3] = {-1, -1, -1};   // per tiling op (SYRK, SQ, X update): -1 = tuned, else this tile configuration
  bool gram_blocks = true;      // schedule "auto": Gram blocks (Eq. 4) on wide buckets; false = plain X iteration
  bool fuse = true;             // a6 / the bf16 NS output fused into the last X-update epilogue (aligned buckets)
  bool keep_o = false;          // keep every matrix's unrounded NS result readable after the call
                                // (dmuon_read_ns_output): fused epilogues also store it, buckets do not share memory
  size_t chunk_bytes = 12ull << 30;   // workspace a bucket may use; larger buckets run as chunks of fewer matrices
  int host_groups = 32;         // dmuon_muon_step_host: at most this many groups of whole shape periods (layers) ...
  int host_slots = 4;           // ... moving through this many device staging slots (measured: profiles/r2_experiments.md)
  int program = 2;              // option "program": run a bucket's whole NS program in ONE launch (ns_program_kernel: products
                                // chained by per-matrix completion counters, matrices in L2-sized groups): 0 = never,
                                // 1 = every eligible bucket (m_pad >= 256, <= 32 products), 2 = "auto": m_pad >= 2048
  size_t l2_group_bytes = 64ull << 20;   // option "l2_group_mb": buffers of one group of matrices in the program kernel
  bool small_fused = true;      // buckets of 256 x 256 (padded) matrices: all NS steps in ONE on-chip launch (ns_small_sm100.cu)
  float tune_ms = 40.f;         // autotune: back-to-back time per candidate (long enough for the power cap to act)
};

// How a matrix is held in the workspace.
enum MatKind : int {
  K_WIDE = 0,      // rows <= cols, both multiples of 128: X [rows x cols] as stored; products SYRK, BX
  K_TALL = 1,      // rows >  cols, both multiples of 128: Y = X^T [rows x cols] AS STORED; products SYRK_T, XB
  K_GENERIC = 2    // any other shape (and every matrix in fp32 check mode): oriented (m <= n, transposed on the way in
                   // and out by the elementwise kernels when rows > cols) and zero-padded to multiples of 128
};

struct MatrixInfo {
  int rows, cols;        // stored
  int m, n;              // oriented (m <= n)
  int m_pad, n_pad;      // padded to multiples of 128
  int kind;              // MatKind
  int buf_rows, buf_cols;// shape of the two X buffers: stored shape (aligned kinds) or m_pad x n_pad (generic)
  bool transposed;       // generic and rows > cols
  int bucket;            // index into Plan::buckets
  int slot;              // position inside its bucket
  int rec;               // index of its MatRec (records are ordered bucket by bucket)
  bool gram;             // bucket eligible for Gram blocks (wide enough that they save work)
  float xscale, gscale;  // powers of two: the workspace holds xscale * X and gscale * G (fp16 range)
};

// Tile configuration of one op of one bucket ("variant" of dmuon_ns_gemm).
struct TileConfig {
  bool pair = false;     // CTA-pair tiling: 256 x 256 units on two SMs (cta_group::2)
  int width = 2;         // single-CTA tiling, blocks per work unit: 2 -> UMMA N = 256, 1 -> N = 128
  int order = 0;         // 0: column-panel-major (all block rows of one column panel first), 1: row-major
  int epi_warps = 4;     // epilogue warps per CTA; 8 (pair tiling only) = two per TMEM lane quarter, for short contractions
};
// Variants 0..3: single CTA, (width, order) = (2,0), (1,0), (2,1), (1,1); 4, 5: CTA pair, order 0, 1; 6, 7: CTA pair
// with 8 epilogue warps, order 0, 1.  The symmetric ops have one ordering: their variants are 0, 1, 4 and 6.
constexpr int kNumVariants = 8;
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

// How a launch's (alpha, beta, beta2) follow from the per-step coefficients (a_i, b_i, c_i) and the bucket's scales
// (the workspace holds cx X and g G, powers of two).
enum CoefKind : int {
  CK_GRAM = 0,   // alpha = g / cx^2                                     SYRK: g G = (g / cx^2) (cx X)(cx X)^T
  CK_POLY,       // alpha = c_s1 / g^2, beta = b_s1 / g                  B = b G + c G G  from g G
  CK_A,          // alpha = 1, beta = a_s1                               T = a G + B G ; G' = a T + T B  (linear in g G)
  CK_RACC,       // alpha = 1, beta = prod a_[s0, s1), beta2 = a_s1      R' = (prod a) B' + a R + B' R
  CK_APOW        // alpha = 1, beta = prod a_[s0, s1]                    X' = (prod a) X + R X           (linear in cx X)
};
struct NsLaunch {
  GemmOp op;
  CoefKind ck;
  int s0, s1;                  // step indices the coefficients come from
  GemmProblem* probs;          // device, one per matrix slot of the bucket shape
  std::string name;            // profiling name: family[m_pad x n_pad]
};
struct NsProgram {
  std::vector<NsLaunch> launches;
  int x_updates = 0;           // how many times X switched buffers (result parity)
};

// Everything the buckets of one (m_pad, n_pad, kind) share: buckets that are chunks of one shape use the same
// workspace slots, so the same problem tables, tile units and tuned variants serve all of them.
struct ShapeTables {
  int m_pad = 0, n_pad = 0, kind = K_WIDE;
  bool gram = false;
  int slots = 0;                       // matrices per chunk (problems per table)
  int buf_rows = 0, buf_cols = 0;
  size_t mat_bytes = 0;                // workspace bytes per matrix slot
  size_t off_p = 0, off_q = 0;         // offsets of the two X buffers inside a slot
  size_t off_sq[5] = {0, 0, 0, 0, 0};  // m_pad x m_pad buffers: G, B, and (Gram-block buckets only) B', T, R
  size_t base = 0;                     // offset of slot 0 in the workspace
  float xscale = 1.f, gscale = 1.f;
  std::map<std::string, NsProgram> programs;   // by partition signature, e.g. "32"
  TileUnit* units[3] = {nullptr, nullptr, nullptr};   // per tiling op (SYRK*, SQ / SQ2, X update)
  int units_per_problem[3] = {0, 0, 0};
  int variant[3] = {0, 0, 0};
  GemmProblem* tune_probs[3] = {nullptr, nullptr, nullptr};   // scratch problem tables for the autotuner
  TileUnit* prog_units[3] = {nullptr, nullptr, nullptr};   // CTA-pair unit tables of the program kernel
  int prog_upp[3] = {0, 0, 0};
  uint32_t* d_done = nullptr;          // [slots] completion counters of the program kernel
  bool onchip = false;                 // m_pad = n_pad = 256: eligible for the on-chip kernel (option small_fused)
  CUtensorMap tm_x0;                   // ... its 3-D map {cols, rows, slot} over the slots' X0 buffers (buffer Q)
  bool tuned_now = false;              // at least one op was timed (not cached) when this plan was built
};

struct BucketPlan {
  int shape = 0;                       // index into Plan::shapes_tbl
  std::vector<int> mats;               // matrix indices (caller order); slot k holds mats[k]
  int rec0 = 0;                        // first MatRec of the bucket
  ElemTables tables{};                 // work lists of the bucket's elementwise launches
  double work = 0;
};

struct Plan {
  std::vector<int32_t> shapes;         // key
  bool fp32 = false;
  bool keep_o = false;
  size_t chunk_bytes = 0;
  int device = 0;
  void* ext_ws = nullptr;
  uint64_t stamp = 0;                  // last use (LRU eviction)
  bool captured = false;               // a CUDA graph recorded a call on this plan: tables re-uploaded at every call, plan and workspace pinned
  uint64_t id = 0;                     // unique; find_plan(id) tells whether the plan still exists
  bool o_valid = false;                // the last call left every matrix's NS result readable in the workspace
  std::vector<MatrixInfo> mats;
  std::vector<ShapeTables> shapes_tbl;
  std::vector<BucketPlan> buckets;     // in execution order
  size_t ws_bytes = 0;
  uint8_t* ws = nullptr;               // device workspace (the device's shared region, or the caller's)
  // elementwise records, ordered bucket by bucket
  std::vector<MatRec> h_recs;          // host mirror (pointers patched per call, uploaded through a pinned snapshot)
  MatRec* d_recs = nullptr;
  float* d_inv_norm = nullptr;
  int bound_kind = -1;                 // what rec.O was last bound for
  std::string bound_key;
  std::vector<void*> d_allocs;         // everything to cudaFree
  int sm_count = 148;
  double tune_seconds = 0;             // time spent measuring tile configurations while building this plan
  ~Plan();
};

size_t plan_workspace_bytes(const int32_t* shapes, int count, const Options& opt);
// Builds (or fetches) the plan for a shape set on the current device.  ext_ws/ext_bytes: caller workspace or (nullptr, 0).
int get_plan(const int32_t* shapes, int count, const Options& opt, void* ext_ws, size_t ext_bytes, cudaStream_t stream,
             Plan** out);
void drop_plans();
int captured_plans();                 // plans a CUDA graph refers to (all devices)
void forget_captures();               // the caller states that every such graph has been destroyed
Plan* find_plan(uint64_t id);
void release_workspaces();
int tune_cache_entries();
void forget_tune_cache();

// What the last X update of a bucket does besides (or instead of) storing the new X.
struct FinalEpilogue {
  Epilogue epi = EPI_F16;
  float lr = 0.f, lrwd = 0.f;
  bool store_c = true;
};
// Enqueue k NS steps of one bucket; X0 is in buffer Q.  result_parity(...) tells where the result ends (0 = Q, 1 = P).
int run_ns_bucket(Plan& plan, int bucket, int steps, const float* coeffs, bool per_step, const Options& opt,
                  const FinalEpilogue& fin, cudaStream_t stream);
int result_parity(const Plan& plan, const ShapeTables& st, int steps, const float* coeffs, bool per_step, const Options& opt);
bool bucket_fuses(const Plan& plan, const ShapeTables& st, int steps, const Options& opt);
// The bucket shape runs its NS steps in the on-chip small-matrix kernel (one launch, nothing stored between products).
bool bucket_onchip(const Plan& plan, const ShapeTables& st, int steps, const Options& opt);
// The bucket shape runs its NS program in the one-launch program kernel (option "program").
bool bucket_program(const Plan& plan, const ShapeTables& st, size_t num_launches, const Options& opt);
size_t program_launches(const Partition& part);      // products of a block schedule: per block of L steps 3 + 4 (L - 1)
std::string partition_key(const Partition& p);

// Build tile units for an op.
std::vector<TileUnit> make_units(GemmOp op, int m_blocks, int n_blocks, const TileConfig& cfg);
int encode_tmap_2d(CUtensorMap* out, const void* base, uint64_t rows, uint64_t cols, uint32_t box_cols,
                   uint32_t box_rows, CUtensorMapSwizzle swizzle = CU_TENSOR_MAP_SWIZZLE_128B);
// A, B: operand matrices with their (rows, cols) as laid out in memory.
int fill_problem(GemmProblem& g, GemmOp op, const void* a_mat, uint64_t a_rows, uint64_t a_cols, const void* b_mat,
                 uint64_t b_rows, uint64_t b_cols, const void* d, void* c, int ldc, const void* d2 = nullptr, int rec = 0);
int check_device();

// ---------------------------------------------------------------- owner assignment (assign.cu)
struct AssignInput {
  int num_shapes, num_ranks;
  const int32_t* counts;        // [num_shapes] n_s
  const int32_t* num_batches;   // [num_shapes] |B_s|
  const int32_t* batch_sizes;   // concatenated B_s
  const double* costs;          // concatenated c_{s,b}
};
int assign_owners_greedy(const AssignInput& in, int32_t* x_out, double* makespan);
int assign_owners_exact(const AssignInput& in, int32_t* x_out, double* makespan, long long node_limit);

}  // namespace dmuon
