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

// ---------------------------------------------------------------- GEMM family (gemm_sm100.cu)
// Tile geometry: output tiles are built from 128 x 128 blocks.  A work unit of the single-CTA tiling is one block row
// of 1 or 2 blocks (UMMA 128 x 128 or 128 x 256); a work unit of the CTA-pair tiling is 2 x 2 blocks (UMMA 256 x 256
// over two SMs).  The contraction advances 64 elements per pipeline stage.
constexpr int kBlk = 128;     // block edge (UMMA_M)
constexpr int kBlkK = 64;     // K elements per stage = one 128-byte swizzle row of fp16

// OP_SYRK  C = alpha A B^T                      (symmetric result: upper blocks computed, mirrored)
// OP_SQ    C = alpha A B^T + beta D             (symmetric result)
// OP_BX    C = alpha A B   + beta D             (B operand MN-major; general result)
// OP_SQ2   C = alpha A B^T + beta D + beta2 D2  (symmetric result; the product of the P_i of a Gram block)
enum GemmOp : int { OP_SYRK = 0, OP_SQ = 1, OP_BX = 2, OP_SQ2 = 3 };
constexpr int kNumOps = 4;

// One problem of a grouped launch.  Lives in device memory; the tensor maps are read by the TMA unit.
struct alignas(128) GemmProblem {
  CUtensorMap tmA;      // operand A: [rows, K] K-major, box {64, 128}
  CUtensorMap tmB;      // operand B: K-major box {64, 128} (SYRK, SQ) or MN-major box {64 (n), 64 (k)} (BX)
  const __half* D;      // addend matrix (SQ: A, BX: X), same leading dimension as C; null for SYRK
  __half* C;            // output
  const __half* D2;     // second addend (SQ2 only)
  int32_t ldc;          // leading dimension of C, D and D2, in elements
  int32_t pad_[25];
};
static_assert(sizeof(GemmProblem) == 384, "GemmProblem layout");

// One work unit of a problem.  Single-CTA tiling: block row, first block column, number of blocks (1 or 2), in
// 128-blocks.  CTA-pair tiling: m_blk, n_blk index 256 x 256 units (width unused).  CTA-quad tiling: two 256 x 256
// units, (m_blk, n_blk) for pair 0 and (width, flags) for pair 1, sharing a block row or a block column (both equal:
// pair 1 shadows pair 0 and stores nothing -- the odd unit left over).
struct TileUnit {
  int16_t m_blk, n_blk, width, flags;
};

struct GemmLaunch {
  GemmOp op;
  const GemmProblem* problems;  // device
  const TileUnit* units;        // device, units_per_problem entries
  int units_per_problem;
  int num_problems;
  int k_blocks;                 // K / 64
  int m_blocks, n_blocks;       // extent of the output in 128-blocks
  bool pair;                    // CTA-pair (cta_group::2) tiling
  bool quad = false;            // CTA quad: two pairs sharing one operand panel by TMA multicast (units hold both)
  float alpha, beta, beta2;
  int grid;                     // CTAs (<= #SM)
};
int launch_ns_gemm(const GemmLaunch& L, cudaStream_t stream);
int gemm_smem_bytes();

// fp32 SIMT check-mode GEMMs (gemm_check.cu): same three ops on fp32 matrices, one problem per launch.
int launch_check_gemm(GemmOp op, const float* in0, const float* in1, float* out, int m, int n, float alpha,
                      float beta, cudaStream_t stream);

// ---------------------------------------------------------------- elementwise family (elementwise.cu)
// Per-matrix record used by every elementwise kernel (device array).
struct MatRec {
  void* W;              // bf16 parameter (muon) / in-out matrix (ns)
  const void* G;        // bf16 gradient (muon)
  void* M;              // bf16 momentum (muon)
  float* W32;           // fp32 master copy of W (dmuon_muon_step_master) or null
  void* U;              // bf16 staging of U, rows*cols, stored orientation (muon); unused (ns)
  void* X0;             // internal buffer receiving the normalised, oriented, padded X0 (fp16 or fp32)
  const void* O;        // internal buffer holding NS_k(X0), oriented + padded
  int32_t rows, cols;   // stored shape
  int32_t m_pad, n_pad; // oriented, padded shape of the internal buffers (leading dimension n_pad)
  int32_t transposed;   // rows > cols
  float scale;          // sqrt(max(1, rows/cols))
  int64_t flat_chunk0;  // first chunk id of this matrix in the flat (momentum / sumsq) chunking
  int64_t tile0;        // first tile id of this matrix in the stored-orientation 64 x 64 tiling
  int64_t ptile0;       // first tile id in the padded, oriented 64 x 64 tiling
};

constexpr int kFlatChunk = 8192;   // elements per flat chunk (one CTA pass)
constexpr int kTile = 64;          // edge of the 2-D elementwise tiles

struct ElemTables {
  const MatRec* recs;          // device [count]
  const int64_t* flat_prefix;  // device [count + 1] chunk prefix
  const int64_t* tile_prefix;  // device [count + 1] stored-orientation tile prefix
  const int64_t* ptile_prefix; // device [count + 1] padded oriented tile prefix
  // Fast paths of the normalise / apply passes (fp16 workspace only).  A matrix is on exactly one path; the other
  // paths' prefix arrays give it zero work items.
  const int64_t* fa_prefix;    // path A: not transposed, rows and cols multiples of 128 (workspace layout == stored
                               //         layout): flat 8192-element chunks
  const int64_t* fb_prefix;    // path B: transposed, rows and cols multiples of 128: 64 x 64 tiles, 16-bit transpose
  int count;
  int64_t flat_chunks, tiles, ptiles, fa_chunks, fb_tiles;
  float* partials;             // device [flat_chunks] per-chunk sum of squares
  float* inv_norm;             // device [count] 1 / (||U||_F + eps)
};

int launch_fill_scratch(void* ptr, size_t bytes, cudaStream_t s);            // autotune operands
int launch_momentum(const ElemTables& T, float mu, cudaStream_t s);          // a1 + a2 partials
int launch_sumsq(const ElemTables& T, cudaStream_t s);                       // a2 alone (ns_batched)
int launch_finalize_norms(const ElemTables& T, float eps, cudaStream_t s);
int launch_normalize(const ElemTables& T, bool from_user, bool fp32_internal, cudaStream_t s);
int launch_apply(const ElemTables& T, float lr, float wd, bool fp32_internal, bool master, cudaStream_t s);   // a6
int launch_store_ns(const ElemTables& T, bool fp32_internal, cudaStream_t s);                    // ns_batched output

int launch_export(const void* O, float* out, int rows, int cols, int n_pad, bool transposed, bool fp32_internal,
                  cudaStream_t s);                                                               // test hook

// ---------------------------------------------------------------- profiling (api.cu)
void prof_begin(const char* name, cudaStream_t s);
void prof_end(cudaStream_t s);
struct ProfScope {
  cudaStream_t s;
  ProfScope(const char* name, cudaStream_t st) : s(st) { prof_begin(name, st); }
  ~ProfScope() { prof_end(s); }
};

}  // namespace dmuon
