// Internal declarations shared by the libdmuon translation units (host side + kernel launchers).
#pragma once

#include <cuda.h>            // CUtensorMap type only; the driver entry point is fetched at run time
#include <cuda_fp16.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include <cstdint>
#include <string>
#include <vector>

#include "../../include/dmuon.h"

namespace dmuon {

// ---------------------------------------------------------------- errors
void set_error(const char* fmt, ...);
#define DMUON_CUDA_CHECK(expr)                                                                   \
  do {                                                                                           \
    cudaError_t _e = (expr);                                                                     \
    if (_e != cudaSuccess) {                                                                     \
      ::dmuon::set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e), __FILE__, __LINE__); \
      return DMUON_ERR_CUDA;                                                                     \
    }                                                                                            \
  } while (0)

constexpr int kMaxDevices = 16;   // per-device state tables (kernel attributes, workspaces)

// ---------------------------------------------------------------- GEMM family (gemm_sm100.cu)
// Tile geometry: output tiles are built from 128 x 128 blocks.  A work unit of the single-CTA tiling is one block row
// of 1 or 2 blocks (UMMA 128 x 128 or 128 x 256); a work unit of the CTA-pair tiling is 2 x 2 blocks (UMMA 256 x 256
// over two SMs).  The contraction advances 64 elements per pipeline stage.
constexpr int kBlk = 128;     // block edge (UMMA_M)
constexpr int kBlkK = 64;     // K elements per stage = one 128-byte swizzle row of fp16

// Products of the Gram-form NS step.  "wide" matrices (rows <= cols) are held as X [m x n]; "tall"
// aligned matrices (rows > cols) are held AS STORED, Y = X^T [n x m], and use the two *_T / XB products, so that no
// transposed copy of a tall matrix is ever made (PAPER.md:174 only asks that the Gram matrix be the small one).
//   OP_SYRK    C = alpha A A^T                      A = X  [m x n] K-major                      (symmetric result)
//   OP_SQ      C = alpha A B^T + beta D             A, B [m x m] K-major, symmetric result
//   OP_BX      C = alpha A B   + beta D             A = R [m x m] K-major, B = D = X [m x n] MN-major; general result
//   OP_SQ2     C = alpha A B^T + beta D + beta2 D2  symmetric result (running product of the P_i of a Gram block)
//   OP_SYRK_T  C = alpha Y^T Y                      Y [n x m]: both operands MN-major             (symmetric result)
//   OP_XB      C = alpha A B^T + beta D             A = D = Y [n x m] K-major, B = R [m x m] (R = R^T); general result
enum GemmOp : int { OP_SYRK = 0, OP_SQ = 1, OP_BX = 2, OP_SQ2 = 3, OP_SYRK_T = 4, OP_XB = 5 };
constexpr int kNumOps = 6;

// What the epilogue does with x = alpha acc + beta D (+ beta2 D2), all in fp32 on the accumulator:
//   EPI_F16           C = fp16(x)
//   EPI_BF16          out = bf16(x / c)                               the last X update of dmuon_ns_batched
//   EPI_APPLY         W' = bf16(W - (lr scale x / c + lr wd W))       the last X update of dmuon_muon_step: step a6
//   EPI_APPLY_MASTER  W32' = W32 - (...), W' = bf16(W32')             (Eq. 1) fused into its epilogue
// For the last three, C may also be written (fp16(x), the unrounded NS result kept for dmuon_read_ns_output).
enum Epilogue : int { EPI_F16 = 0, EPI_BF16 = 1, EPI_APPLY = 2, EPI_APPLY_MASTER = 3 };
constexpr int kNumEpi = 4;

// One problem of a grouped launch.  Lives in device memory; the tensor maps are read by the TMA unit.
struct alignas(128) GemmProblem {
  CUtensorMap tmA;      // operand A: K-major box {64 (k), 128 (rows)}; MN-major (SYRK_T) box {64 (m), 64 (k)}
  CUtensorMap tmB;      // operand B: K-major box {64, 128}; MN-major (BX, SYRK_T) box {64 (n), 64 (k)}
  CUtensorMap tmC;      // output C (fused epilogues write it only when the launch says store_c): box {32 (cols), 32 (rows)},
                        // 64-byte swizzle -- the epilogue warps' staging tiles; the mirrored tile of a symmetric result
                        // goes out through the same map at the transposed coordinates
  CUtensorMap tmD;      // addend D (SQ: A, BX / XB: X), same shape and boxes as C; unused for SYRK
  CUtensorMap tmD2;     // second addend (SQ2 only)
  int32_t ldc;          // leading dimension of C (and of W / W32 in the fused epilogues), in elements
  int32_t rec;          // index of the matrix's MatRec (fused epilogues read W / W32 / scale there)
  int32_t pad_[30];
};
static_assert(sizeof(GemmProblem) == 768, "GemmProblem layout");

// One work unit of a problem.  Single-CTA tiling: block row, first block column, number of blocks (1 or 2), in
// 128-blocks.  CTA-pair tiling: m_blk, n_blk index 256 x 256 units (width unused).
struct TileUnit {
  int16_t m_blk, n_blk, width, flags;
};

struct MatRec;

struct GemmLaunch {
  GemmOp op;
  Epilogue epi = EPI_F16;
  const GemmProblem* problems;  // device
  const TileUnit* units;        // device, units_per_problem entries
  const MatRec* recs = nullptr; // device (fused epilogues)
  int units_per_problem;
  int num_problems;
  int k_blocks;                 // K / 64
  int m_blocks, n_blocks;       // extent of the output in 128-blocks (rows, columns)
  bool pair;                    // CTA-pair (cta_group::2) tiling
  int epi_warps = 4;            // epilogue warps per CTA: 4, or 8 (CTA-pair tiling only)
  float alpha, beta, beta2;
  float lr = 0.f, lrwd = 0.f;   // EPI_APPLY*: learning rate and lr * wd
  bool store_c = true;          // fused epilogues: also store fp16(x) to C
  int rec_base = 0;             // MatRec of problem p = recs[rec_base + problems[p].rec]
  int grid;                     // CTAs (<= #SM)
};
int launch_ns_gemm(const GemmLaunch& L, cudaStream_t stream);
int gemm_smem_bytes();

// The whole NS program of a bucket in ONE launch (gemm_sm100.cu, ns_program_kernel): products chained by per-matrix
// completion counters, matrices taken in L2-sized groups.  CTA-pair tiling; aligned wide / tall and generic buckets with
// m_pad >= 256.
constexpr int kMaxProgPhases = 32;
struct ProgPhaseHost {
  GemmOp op;
  const GemmProblem* probs;     // device: one problem per slot of the bucket shape
  float alpha, beta, beta2;
};
struct ProgLaunch {
  ProgPhaseHost ph[kMaxProgPhases];
  int num_phases = 0;
  bool tall = false;            // SYRK_T / XB (a tall matrix held as stored) instead of SYRK / BX
  Epilogue final_epi = EPI_F16; // epilogue of the last phase (an X update)
  const TileUnit* units[3];     // CTA-pair unit tables per tiling op (Gram product, m x m products, X update)
  int upp[3];
  const MatRec* recs = nullptr;
  int rec_base = 0;
  int count = 0;                // matrices (slots 0 .. count - 1)
  int group = 1;                // matrices per L2-resident group
  int m_blocks = 0, n_blocks = 0;   // oriented padded shape in 128-blocks
  uint32_t* done = nullptr;     // device [count + 1]: completion counters and the unit queue (zeroed by the launcher)
  float lr = 0.f, lrwd = 0.f;
  bool store_c = true;
  int grid = 148;
};
int launch_ns_program(const ProgLaunch& L, cudaStream_t stream);

// On-chip NS of small matrices (ns_small_sm100.cu): all k steps of every 256 x 256 (padded) matrix of a bucket in ONE
// launch, X / G / B resident in the shared memory of a CTA pair (PAPER.md:170 Gram form, :180 batching by shape).
constexpr int kSmallEdge = 256;        // m_pad = n_pad = 256
constexpr int kSmallMaxSteps = 16;
struct SmallLaunch {
  const CUtensorMap* tmX;      // host copy of the 3-D map {256 cols, 256 rows, slots} over the bucket's X0 buffers
  void* out;                   // fp16 X_k of slot s at out + s * slot_bytes (row stride 256); written for EPI_F16 or store_c
  size_t slot_bytes;
  const MatRec* recs = nullptr;
  int rec_base = 0;
  int count = 0;               // matrices (slots 0 .. count - 1)
  int steps = 0;
  float gram_alpha = 1.f;      // G~ = gram_alpha X~ X~^T
  float poly_alpha[kSmallMaxSteps], poly_beta[kSmallMaxSteps];   // B = poly_beta G~ + poly_alpha G~ G~
  float x_beta[kSmallMaxSteps];                                   // X~' = x_beta X~ + B X~
  Epilogue epi = EPI_F16;      // what the last X update does (see Epilogue)
  float lr = 0.f, lrwd = 0.f;
  bool store_c = true;
  int grid = 148;
};
int launch_ns_small(const SmallLaunch& L, cudaStream_t stream);

// fp32 SIMT check-mode GEMMs (gemm_check.cu): same three ops on fp32 matrices, one problem per launch.
int launch_check_gemm(GemmOp op, const float* in0, const float* in1, float* out, int m, int n, float alpha,
                      float beta, cudaStream_t stream);

// ---------------------------------------------------------------- elementwise family (elementwise.cu)
// Per-matrix record used by every elementwise kernel and by the fused GEMM epilogues (device array).
struct MatRec {
  void* W;              // bf16 parameter (muon) / in-out matrix (ns)
  const void* G;        // bf16 gradient (muon)
  void* M;              // bf16 momentum (muon)
  float* W32;           // fp32 master copy of W (dmuon_muon_step_master) or null
  void* U;              // bf16 staging of U, rows*cols, stored orientation (muon); unused (ns)
  void* X0;             // internal buffer receiving the normalised, scaled, padded X0 (fp16 or fp32)
  const void* O;        // internal buffer holding NS_k(X0) (scaled by xscale)
  int32_t rows, cols;   // stored shape
  int32_t m_pad, n_pad; // shape of the internal buffers: [m_pad x n_pad], leading dimension n_pad.  Generic matrices:
                        // oriented (m <= n) and padded to 128; aligned matrices: the stored shape itself
  int32_t transposed;   // internal buffer = transpose of the stored matrix (generic tall matrices only)
  float scale;          // sqrt(max(1, rows/cols))                       (reading N4)
  float xscale;         // power of two c: the internal buffers hold c X  (fp16 range)
  float inv_xscale;     // 1 / c (exact)
  int64_t flat_chunk0;  // first chunk id of this matrix in the flat (momentum / sumsq) chunking
  int64_t tile0;        // first tile id of this matrix in the stored-orientation 64 x 64 tiling
  int64_t ptile0;       // first tile id in the padded, oriented 64 x 64 tiling
};

constexpr int kFlatChunk = 8192;   // elements per flat chunk (one CTA pass)
constexpr int kTile = 64;          // edge of the 2-D elementwise tiles

// Work lists of one elementwise launch: the matrices of ONE bucket (the other matrices of the plan have no work items).
struct ElemTables {
  const MatRec* recs;          // device [count] (all matrices of the plan)
  const int64_t* flat_prefix;  // device [count + 1] chunk prefix
  const int64_t* tile_prefix;  // device [count + 1] stored-orientation tile prefix   (generic matrices)
  const int64_t* ptile_prefix; // device [count + 1] padded oriented tile prefix      (generic matrices)
  const int64_t* fa_prefix;    // device [count + 1] flat chunk prefix (aligned matrices: internal layout == stored layout)
  int count;
  int64_t flat_chunks, tiles, ptiles, fa_chunks;
  float* partials;             // device [flat_chunks] per-chunk sum of squares
  float* inv_norm;             // device [count] xscale / (||U||_F + eps)
};

int launch_fill_scratch(void* ptr, size_t bytes, cudaStream_t s);            // autotune operands
int launch_momentum(const ElemTables& T, float mu, bool exact, cudaStream_t s);   // a1 + a2 partials (exact: fp64 decisions)
int launch_sumsq(const ElemTables& T, cudaStream_t s);                       // a2 alone (ns_batched)
int launch_finalize_norms(const ElemTables& T, float eps, cudaStream_t s);
int launch_normalize(const ElemTables& T, bool from_user, bool fp32_internal, cudaStream_t s);
int launch_apply(const ElemTables& T, float lr, float wd, bool fp32_internal, bool master, cudaStream_t s);   // a6 (not fused)
int launch_store_ns(const ElemTables& T, bool fp32_internal, cudaStream_t s);                    // ns_batched output (not fused)

// Non-matrix parameters (Alg. 1 l.16): decoupled AdamW, one flat launch over all tensors.
struct AdamRec {
  void* p;              // bf16 parameter, updated in place
  const void* g;        // bf16 gradient
  float* m;             // fp32 first moment
  float* v;             // fp32 second moment
  int64_t numel;
};
struct AdamScalars {
  float lr, beta1, beta2, eps, wd;
  float inv_bc1;        // 1 / (1 - beta1^t)
  float inv_sqrt_bc2;   // 1 / sqrt(1 - beta2^t)
};
int launch_adamw(const AdamRec* d_recs, const int64_t* d_prefix, int count, int64_t total_chunks, const AdamScalars& sc,
                 cudaStream_t s);
// The same kernel with its work table in a static device array instead of cudaMalloc'ed memory (elementwise.cu):
// builds and uploads the table of this call, then launches.  At most kAdamStaticMaxTensors tensors per call.
constexpr int kAdamStaticMaxTensors = DMUON_ADAMW_NOALLOC_MAX_TENSORS;       // dmuon.h
int launch_adamw_static(void* const* params, const void* const* grads, void* const* exp_avg, void* const* exp_avg_sq,
                        const int64_t* numel, int count, const AdamScalars& sc, cudaStream_t s);

int launch_export(const void* O, float* out, int rows, int cols, int n_pad, bool transposed, bool fp32_internal,
                  float inv_xscale, cudaStream_t s);                                             // test hook

// ---------------------------------------------------------------- profiling (api.cu)
void prof_begin(const char* name, cudaStream_t s);
void prof_end(cudaStream_t s);
struct ProfScope {
  cudaStream_t s;
  ProfScope(const char* name, cudaStream_t st) : s(st) { prof_begin(name, st); }
  ~ProfScope() { prof_end(s); }
};

}  // namespace dmuon
