// Persistent grouped GEMM family for the Gram-form Newton-Schulz step on sm_100a (steps a3, a4, a5 of DESIGN.md):
//
//   OP_SYRK  C = alpha * X X^T                (PAPER.md:170 G = X X^T; symmetric kernel of PAPER.md:182)
//   OP_SQ    C = alpha * A A + beta * A       (the polynomial in the Gram matrix; A A = A A^T)
//   OP_BX    C = alpha * B X + beta * X       (X_{i+1} = P X_i with the a X term in the epilogue)
//   OP_SQ2   C = alpha * A B + beta * D + beta2 * D2   (symmetric, two addends: the running product of the
//                                              P_i = a_i I + B_i of a Gram block, Eq. 4)
//
// Two tilings of the same warp-specialised pipeline (warp 0 = TMA producer, warp 1 = tcgen05.mma issuer and TMEM
// owner, warps 2..5 = epilogue: TMEM -> registers -> global):
//
//   single CTA  (cta_group::1)  one CTA per SM computes a 128 x 128 or 128 x 256 unit; 4-stage ring of 48 KB.
//   CTA pair    (cta_group::2)  a cluster of two CTAs (one TPC) computes a 256 x 256 unit with UMMA M = 256, N = 256:
//                               each CTA stages its 128 rows of operand A and its 128 columns of operand B (32 KB per
//                               stage, 6 stages) and holds its 128 accumulator rows in its own TMEM, so a unit moves
//                               2/3 of the L2->SMEM bytes per FLOP of the single-CTA tiling.  The leader CTA issues the
//                               MMAs; both producers signal the leader's "full" barrier; tcgen05.commit multicasts the
//                               "slot free" and "accumulator ready" arrivals to both CTAs.
//
// Operands are fp16, 128-byte-swizzled tiles moved by cp.async.bulk.tensor; accumulators are fp32 in TMEM, two
// of them (2 x 256 columns) so the epilogue of one unit overlaps the mainloop of the next.  The symmetric ops visit
// only upper-triangular blocks and store each off-diagonal 128 x 128 block twice (direct and mirrored), so the dense
// output later steps need is kept.
#include "common.h"
#include "umma.cuh"

namespace dmuon {
namespace {

using namespace umma;

constexpr int kBlockBytes = kBlk * kBlkK * 2;   // 16 KB: 128 rows x 128 B of one operand block
constexpr int kNumThreads = 192;
constexpr int kTmemCols = 512;
constexpr int kAccCols = 256;                   // columns per accumulator stage
constexpr int kMaxStages = 6;

template <bool kPair> struct Tiling;
template <> struct Tiling<false> {              // one CTA: A block + up to two B blocks per stage
  static constexpr int kStages = 4;
  static constexpr int kStageBytes = 3 * kBlockBytes;
};
template <> struct Tiling<true> {               // CTA pair: this CTA's A block + its B block per stage
  static constexpr int kStages = 6;
  static constexpr int kStageBytes = 2 * kBlockBytes;
};

struct SmemCtl {
  uint64_t full[kMaxStages];
  uint64_t empty[kMaxStages];
  uint64_t tmem_full[2];
  uint64_t tmem_empty[2];
  uint32_t tmem_base;
  uint32_t pad;
};
static_assert(sizeof(SmemCtl) <= 256, "SmemCtl");
template <bool kPair> constexpr int smem_bytes() {
  return Tiling<kPair>::kStages * Tiling<kPair>::kStageBytes + 1024 /*alignment slack*/ + 256 /*SmemCtl*/;
}

// ------------------------------------------------------------------------------------------------ epilogue
// Addend words of one 32-column chunk of one row: 64 bytes of D (and of D2 for OP_SQ2).  Loaded one chunk ahead of the
// arithmetic (two register sets, alternating) so that their L2 latency overlaps the TMEM load and the stores of the
// previous chunk: with short contractions (K <= 1024) the epilogue, not the mainloop, sets the pace.
struct Addends {
  uint4 d[4];
  uint4 e[4];
};
template <int kOp>
__device__ __forceinline__ void load_addends(Addends& a, const __half* __restrict__ D, const __half* __restrict__ D2,
                                             int64_t ldc, int64_t grow, int64_t gcol) {
  if (kOp == OP_SYRK) return;
  const uint4* dp = reinterpret_cast<const uint4*>(D + grow * ldc + gcol);
#pragma unroll
  for (int g = 0; g < 4; ++g) a.d[g] = __ldg(dp + g);
  if (kOp == OP_SQ2) {
    const uint4* ep = reinterpret_cast<const uint4*>(D2 + grow * ldc + gcol);
#pragma unroll
    for (int g = 0; g < 4; ++g) a.e[g] = __ldg(ep + g);
  }
}

// One 32-column chunk of one accumulator row: v = 32 fp32 accumulators of row `grow`, columns [gcol, gcol + 32).
template <int kOp>
__device__ __forceinline__ void epilogue_chunk(const uint32_t (&v)[32], const Addends& a, __half* __restrict__ C,
                                               int64_t ldc, int64_t grow, int64_t gcol, float alpha, float beta,
                                               float beta2, bool mirror) {
  uint32_t o[16];
  if (kOp != OP_SYRK) {
#pragma unroll
    for (int g = 0; g < 4; ++g) {
      const uint32_t dw[4] = {a.d[g].x, a.d[g].y, a.d[g].z, a.d[g].w};
      const uint32_t ew[4] = {a.e[g].x, a.e[g].y, a.e[g].z, a.e[g].w};
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const float2 df = __half22float2(*reinterpret_cast<const __half2*>(&dw[e]));
        float ax = beta * df.x, ay = beta * df.y;
        if (kOp == OP_SQ2) {
          const float2 ef = __half22float2(*reinterpret_cast<const __half2*>(&ew[e]));
          ax = fmaf(beta2, ef.x, ax);
          ay = fmaf(beta2, ef.y, ay);
        }
        const float lo = fmaf(alpha, __uint_as_float(v[g * 8 + e * 2]), ax);
        const float hi = fmaf(alpha, __uint_as_float(v[g * 8 + e * 2 + 1]), ay);
        o[g * 4 + e] = pack_half2(lo, hi);
      }
    }
  } else {
#pragma unroll
    for (int e = 0; e < 16; ++e)
      o[e] = pack_half2(alpha * __uint_as_float(v[2 * e]), alpha * __uint_as_float(v[2 * e + 1]));
  }
  uint4* cp = reinterpret_cast<uint4*>(C + grow * ldc + gcol);
#pragma unroll
  for (int g = 0; g < 4; ++g) cp[g] = make_uint4(o[g * 4], o[g * 4 + 1], o[g * 4 + 2], o[g * 4 + 3]);
  if (kOp != OP_BX && mirror) {
    // mirrored store C[col][row]: for a fixed column the 32 lanes hold 32 consecutive rows -> 64-byte runs
    __half* mp = C + gcol * ldc + grow;
#pragma unroll
    for (int e = 0; e < 16; ++e) {
      const __half2 h = *reinterpret_cast<const __half2*>(&o[e]);
      mp[static_cast<int64_t>(2 * e) * ldc] = __low2half(h);
      mp[static_cast<int64_t>(2 * e + 1) * ldc] = __high2half(h);
    }
  }
}

// ------------------------------------------------------------------------------------------------ the kernel body
// mb, nb: extent of the output in 128-blocks (rows, columns); pair units may overhang it (TMA zero-fills the
// operands there, the epilogue skips those blocks).
template <int kOp, bool kPair>
__device__ __forceinline__ void ns_gemm_body(const GemmProblem* __restrict__ probs, const TileUnit* __restrict__ units,
                                             int units_per_problem, int total_units, int k_blocks, int mb, int nb,
                                             float alpha, float beta, float beta2) {
  constexpr bool kSym = (kOp != OP_BX);
  constexpr bool kBMn = (kOp == OP_BX);
  constexpr int kCG = kPair ? 2 : 1;
  constexpr int kStages = Tiling<kPair>::kStages;
  constexpr int kStageBytes = Tiling<kPair>::kStageBytes;

  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;    // swizzle-128B atoms need 1024-byte alignment
  SmemCtl* ctl = reinterpret_cast<SmemCtl*>(smem_raw + (base - raw) + kStages * kStageBytes);
  const uint32_t ctl_addr = base + kStages * kStageBytes;
  const uint32_t bar_full = ctl_addr + offsetof(SmemCtl, full);
  const uint32_t bar_empty = ctl_addr + offsetof(SmemCtl, empty);
  const uint32_t bar_tfull = ctl_addr + offsetof(SmemCtl, tmem_full);
  const uint32_t bar_tempty = ctl_addr + offsetof(SmemCtl, tmem_empty);

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const uint32_t rank = kPair ? cluster_ctarank() : 0u;          // 0 = leader of the pair
  const int worker = kPair ? (blockIdx.x >> 1) : blockIdx.x;
  const int num_workers = kPair ? (gridDim.x >> 1) : gridDim.x;

  if (threadIdx.x == 0) {
    for (int s = 0; s < kStages; ++s) {
      mbar_init(bar_full + 8 * s, 1);
      mbar_init(bar_empty + 8 * s, 1);
    }
    for (int s = 0; s < 2; ++s) {
      mbar_init(bar_tfull + 8 * s, 1);
      mbar_init(bar_tempty + 8 * s, kPair ? 8 : 4);              // one arrival per epilogue warp (of both CTAs)
    }
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc<kCG>(ctl_addr + offsetof(SmemCtl, tmem_base), kTmemCols);
  tcgen05_fence_before();
  if (kPair) cluster_sync(); else __syncthreads();
  tcgen05_fence_after();
  const uint32_t tmem_base = ctl->tmem_base;

  if (warp == 0) {
    // ================================================================== TMA producer (both CTAs of a pair)
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      for (int u = worker; u < total_units; u += num_workers) {
        const int p = u / units_per_problem;
        const TileUnit tu = units[u - p * units_per_problem];
        const GemmProblem* pr = probs + p;
        const uint64_t tmA = reinterpret_cast<uint64_t>(&pr->tmA);
        const uint64_t tmB = reinterpret_cast<uint64_t>(&pr->tmB);
        // the next unit of this worker usually belongs to another matrix: fetch its descriptors ahead of use
        const int un = u + num_workers;
        if (un < total_units) {
          const int pn = un / units_per_problem;
          if (pn != p) {
            tma_prefetch_desc(reinterpret_cast<uint64_t>(&probs[pn].tmA));
            tma_prefetch_desc(reinterpret_cast<uint64_t>(&probs[pn].tmB));
          }
        }
        const int a_blk = kPair ? 2 * tu.m_blk + static_cast<int>(rank) : tu.m_blk;      // this CTA's 128 rows of A
        const int b_blk = kPair ? 2 * tu.n_blk + static_cast<int>(rank) : tu.n_blk;      // its first 128 columns of B
        const int w = kPair ? 1 : tu.width;
        for (int kb = 0; kb < k_blocks; ++kb) {
          mbar_wait(bar_empty + 8 * stage, phase ^ 1);
          const uint32_t sA = base + stage * kStageBytes;
          const uint32_t sB = sA + kBlockBytes;
          if (!kPair) {
            const uint32_t fb = bar_full + 8 * stage;
            mbar_expect_tx(fb, kBlockBytes + w * kBlockBytes);
            tma_load_2d(sA, tmA, kb * kBlkK, a_blk * kBlk, fb);
            if (!kBMn) {
              for (int q = 0; q < w; ++q) tma_load_2d(sB + q * kBlockBytes, tmB, kb * kBlkK, (b_blk + q) * kBlk, fb);
            } else {
              for (int q = 0; q < 2 * w; ++q)   // 64 (n) x 64 (k) boxes, 8 KB each
                tma_load_2d(sB + q * (kBlockBytes / 2), tmB, b_blk * kBlk + q * 64, kb * kBlkK, fb);
            }
          } else {
            // both halves of the stage are accounted on the leader's barrier (its MMA thread waits there)
            if (rank == 0) mbar_expect_tx(bar_full + 8 * stage, 2 * kStageBytes);
            const uint32_t fb = mapa(bar_full + 8 * stage, 0);
            tma_load_2d_pair(sA, tmA, kb * kBlkK, a_blk * kBlk, fb);
            if (!kBMn) {
              tma_load_2d_pair(sB, tmB, kb * kBlkK, b_blk * kBlk, fb);
            } else {
              tma_load_2d_pair(sB, tmB, b_blk * kBlk, kb * kBlkK, fb);
              tma_load_2d_pair(sB + kBlockBytes / 2, tmB, b_blk * kBlk + 64, kb * kBlkK, fb);
            }
          }
          if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
      }
    }
    __syncwarp();
  } else if (warp == 1) {
    // ================================================================== MMA issuer (leader CTA only in a pair)
    if (lane == 0 && rank == 0) {
      int stage = 0;
      uint32_t phase = 0;
      int it = 0;
      for (int u = worker; u < total_units; u += num_workers, ++it) {
        const int p = u / units_per_problem;
        const TileUnit tu = units[u - p * units_per_problem];
        const uint32_t idesc = make_idesc(kPair ? 256 : 128, kPair ? 256 : tu.width * kBlk, kBMn);
        const int as = it & 1;
        const uint32_t aphase = (it >> 1) & 1;
        mbar_wait(bar_tempty + 8 * as, aphase ^ 1);    // epilogue has drained this accumulator
        tcgen05_fence_after();
        const uint32_t d_tmem = tmem_base + as * kAccCols;
        for (int kb = 0; kb < k_blocks; ++kb) {
          mbar_wait(bar_full + 8 * stage, phase);       // TMA bytes have landed (in both CTAs of a pair)
          tcgen05_fence_after();
          const uint32_t sA = base + stage * kStageBytes;
          const uint32_t sB = sA + kBlockBytes;
#pragma unroll
          for (int k = 0; k < kBlkK / 16; ++k) {
            const uint64_t ad = desc_kmajor(sA + k * 32);
            const uint64_t bd = kBMn ? desc_mnmajor(sB + k * 2048) : desc_kmajor(sB + k * 32);
            mma_f16<kCG>(d_tmem, ad, bd, idesc, (kb | k) != 0);
          }
          // frees the smem slot (in both CTAs) when these MMAs finish
          if (kPair) mma_commit_pair(bar_empty + 8 * stage, 3); else mma_commit(bar_empty + 8 * stage);
          if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
        // accumulator complete -> epilogue (of both CTAs)
        if (kPair) mma_commit_pair(bar_tfull + 8 * as, 3); else mma_commit(bar_tfull + 8 * as);
      }
    }
    __syncwarp();
  } else {
    // ================================================================== epilogue (4 warps, one TMEM lane quarter each)
    const int q = warp & 3;
    const int row = q * 32 + lane;
    const uint32_t tempty_leader = kPair ? mapa(bar_tempty, 0) : bar_tempty;
    int it = 0;
    for (int u = worker; u < total_units; u += num_workers, ++it) {
      const int p = u / units_per_problem;
      const TileUnit tu = units[u - p * units_per_problem];
      const GemmProblem* pr = probs + p;
      __half* __restrict__ C = pr->C;
      const __half* __restrict__ D = pr->D;
      const __half* __restrict__ D2 = pr->D2;
      const int64_t ldc = pr->ldc;
      const int as = it & 1;
      const uint32_t aphase = (it >> 1) & 1;
      const int bi = kPair ? 2 * tu.m_blk + static_cast<int>(rank) : tu.m_blk;      // row block of this CTA
      const int bj0 = kPair ? 2 * tu.n_blk : tu.n_blk;                               // first column block
      const int nbk = kPair ? 2 : tu.width;
      const int64_t grow = static_cast<int64_t>(bi) * kBlk + row;
      const int64_t gcol0 = static_cast<int64_t>(bj0) * kBlk;
      // chunks (32 columns each) this warp stores: inside the matrix and, for symmetric results, not left of the
      // diagonal block (those blocks are written by the mirror of another unit)
      int c_lo = 0, c_hi = 0;
      if (bi < mb) {
        c_lo = (kSym && bi > bj0) ? (bi - bj0) * 4 : 0;
        c_hi = (nb - bj0 < nbk ? nb - bj0 : nbk) * 4;
      }
      Addends a0 = {}, a1 = {};
      if (c_lo < c_hi) load_addends<kOp>(a0, D, D2, ldc, grow, gcol0 + c_lo * 32);   // before the accumulator is ready
      mbar_wait(bar_tfull + 8 * as, aphase);
      tcgen05_fence_after();
      const uint32_t taddr = tmem_base + as * kAccCols + (static_cast<uint32_t>(q * 32) << 16);
      for (int c = c_lo; c < c_hi; c += 2) {
        uint32_t v[32];
        if (c + 1 < c_hi) load_addends<kOp>(a1, D, D2, ldc, grow, gcol0 + (c + 1) * 32);
        tmem_ld_32x32(taddr + c * 32, v);
        tmem_wait_ld();
        epilogue_chunk<kOp>(v, a0, C, ldc, grow, gcol0 + c * 32, alpha, beta, beta2, bj0 + (c >> 2) != bi);
        if (c + 1 < c_hi) {
          if (c + 2 < c_hi) load_addends<kOp>(a0, D, D2, ldc, grow, gcol0 + (c + 2) * 32);
          tmem_ld_32x32(taddr + (c + 1) * 32, v);
          tmem_wait_ld();
          epilogue_chunk<kOp>(v, a1, C, ldc, grow, gcol0 + (c + 1) * 32, alpha, beta, beta2, bj0 + ((c + 1) >> 2) != bi);
        }
      }
      // accumulator fully read by this warp: hand it back to the MMA thread
      tcgen05_fence_before();
      __syncwarp();
      if (lane == 0) {
        if (kPair) mbar_arrive_cluster(tempty_leader + 8 * as); else mbar_arrive(bar_tempty + 8 * as);
      }
    }
  }

  tcgen05_fence_before();
  if (kPair) cluster_sync(); else __syncthreads();
  if (warp == 1) tmem_dealloc<kCG>(tmem_base, kTmemCols);
}

// One named entry point per product and tiling, so profiles (ncu -k) and launch lists tell them apart.
#define DMUON_GEMM_ENTRY(name, op, pair)                                                                        \
  __global__ void __launch_bounds__(kNumThreads, 1)                                                             \
  name(const GemmProblem* __restrict__ probs, const TileUnit* __restrict__ units, int units_per_problem,       \
       int total_units, int k_blocks, int mb, int nb, float alpha, float beta, float beta2) {                   \
    ns_gemm_body<op, pair>(probs, units, units_per_problem, total_units, k_blocks, mb, nb, alpha, beta, beta2); \
  }
DMUON_GEMM_ENTRY(ns_syrk_xxt_kernel, OP_SYRK, false)
DMUON_GEMM_ENTRY(ns_sq_poly_kernel, OP_SQ, false)
DMUON_GEMM_ENTRY(ns_bx_update_kernel, OP_BX, false)
DMUON_GEMM_ENTRY(ns_syrk_xxt_pair_kernel, OP_SYRK, true)
DMUON_GEMM_ENTRY(ns_sq_poly_pair_kernel, OP_SQ, true)
DMUON_GEMM_ENTRY(ns_bx_update_pair_kernel, OP_BX, true)
DMUON_GEMM_ENTRY(ns_gram_acc_kernel, OP_SQ2, false)
DMUON_GEMM_ENTRY(ns_gram_acc_pair_kernel, OP_SQ2, true)
#undef DMUON_GEMM_ENTRY

typedef void (*GemmKernel)(const GemmProblem*, const TileUnit*, int, int, int, int, int, float, float, float);

template <bool kPair>
int launch_op(GemmKernel kern, bool* configured, const GemmLaunch& L, cudaStream_t stream) {
  constexpr int kSmem = smem_bytes<kPair>();
  if (!*configured) {
    DMUON_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmem));
    *configured = true;
  }
  const int total = L.units_per_problem * L.num_problems;
  if (total <= 0) return DMUON_OK;
  const int workers = kPair ? L.grid / 2 : L.grid;
  const int use = workers < total ? workers : total;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(kPair ? 2 * use : use);
  cfg.blockDim = dim3(kNumThreads);
  cfg.dynamicSmemBytes = kSmem;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = kPair ? 2 : 1;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  DMUON_CUDA_CHECK(cudaLaunchKernelEx(&cfg, kern, L.problems, L.units, L.units_per_problem, total, L.k_blocks,
                                      L.m_blocks, L.n_blocks, L.alpha, L.beta, L.beta2));
  return DMUON_OK;
}

}  // namespace

int gemm_smem_bytes() { return smem_bytes<false>() > smem_bytes<true>() ? smem_bytes<false>() : smem_bytes<true>(); }

int launch_ns_gemm(const GemmLaunch& L, cudaStream_t stream) {
  static bool configured[2 * kNumOps] = {};
  if (L.op < OP_SYRK || L.op >= kNumOps) {
    set_error("launch_ns_gemm: bad op %d", static_cast<int>(L.op));
    return DMUON_ERR_INVALID_ARG;
  }
  static const GemmKernel kSingle[kNumOps] = {ns_syrk_xxt_kernel, ns_sq_poly_kernel, ns_bx_update_kernel, ns_gram_acc_kernel};
  static const GemmKernel kPairK[kNumOps] = {ns_syrk_xxt_pair_kernel, ns_sq_poly_pair_kernel, ns_bx_update_pair_kernel,
                                             ns_gram_acc_pair_kernel};
  if (L.pair) return launch_op<true>(kPairK[L.op], &configured[kNumOps + L.op], L, stream);
  return launch_op<false>(kSingle[L.op], &configured[L.op], L, stream);
}

}  // namespace dmuon
