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
#include <cstdio>
#include <cstdlib>

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

// ------------------------------------------------------------------------------------------------ CTA quad
// Cluster of four CTAs = two CTA pairs (ranks 0,1 and 2,3), each pair computing one 256 x 256 unit with
// cta_group::2 MMAs as above; the two units of a quad share one operand panel (same block row: operand A shared;
// same block column: operand B shared), and the shared tiles are fetched from L2 ONCE and multicast by TMA into both
// pairs' shared memories.  The pair tiling reads 128 FLOP per L2->SMEM byte, which is what bounds it (0.87-0.89 of the
// tensor peak at any clock, profiles/r1_step_l4_ncu_full.md); a quad reads 171 FLOP/byte.
//
// Protocol differences to the pair tiling: the bytes landing in a pair's two shared memories are all accounted on that
// pair leader's "full" barrier, whoever sent them (cta_group::2 TMA: unicast loads name the leader's barrier, multicast
// loads name it through the cleared pair bit); "empty" barriers count two arrivals, one tcgen05.commit from each pair
// leader, multicast to all four CTAs, so the quad moves through the ring in lockstep (a multicast may overwrite the
// other pair's slot only when that pair has consumed it too).
constexpr int kQuadThreads = 192;

struct QuadCtl {
  uint64_t full[kMaxStages];
  uint64_t empty[kMaxStages];
  uint64_t tmem_full[2];
  uint64_t tmem_empty[2];
  uint32_t tmem_base;
  uint32_t pad;
};
static_assert(sizeof(QuadCtl) <= 256, "QuadCtl");

template <int kOp>
__device__ __forceinline__ void ns_gemm_quad_body(const GemmProblem* __restrict__ probs,
                                                  const TileUnit* __restrict__ units, int units_per_problem,
                                                  int total_units, int k_blocks, int mb, int nb, float alpha, float beta,
                                                  float beta2) {
  constexpr bool kSym = (kOp != OP_BX);
  constexpr bool kBMn = (kOp == OP_BX);
  constexpr int kStages = Tiling<true>::kStages;
  constexpr int kStageBytes = Tiling<true>::kStageBytes;

  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;
  QuadCtl* ctl = reinterpret_cast<QuadCtl*>(smem_raw + (base - raw) + kStages * kStageBytes);
  const uint32_t ctl_addr = base + kStages * kStageBytes;
  const uint32_t bar_full = ctl_addr + offsetof(QuadCtl, full);
  const uint32_t bar_empty = ctl_addr + offsetof(QuadCtl, empty);
  const uint32_t bar_tfull = ctl_addr + offsetof(QuadCtl, tmem_full);
  const uint32_t bar_tempty = ctl_addr + offsetof(QuadCtl, tmem_empty);

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();          // 0..3
  const uint32_t pair = rank >> 1;                  // which unit of the quad
  const uint32_t half = rank & 1;                   // 0 = leader of the pair
  const uint32_t leader = rank & ~1u;
  const uint16_t pair_mask = static_cast<uint16_t>(3u << leader);
  const int worker = blockIdx.x >> 2;
  const int num_workers = gridDim.x >> 2;

  if (threadIdx.x == 0) {
    for (int s = 0; s < kStages; ++s) {
      mbar_init(bar_full + 8 * s, 1);
      mbar_init(bar_empty + 8 * s, 2);              // one commit from each pair leader
    }
    for (int s = 0; s < 2; ++s) {
      mbar_init(bar_tfull + 8 * s, 1);
      mbar_init(bar_tempty + 8 * s, 8);             // epilogue warps of both CTAs of the pair
    }
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc<2>(ctl_addr + offsetof(QuadCtl, tmem_base), kTmemCols);
  tcgen05_fence_before();
  cluster_sync();
  tcgen05_fence_after();
  const uint32_t tmem_base = ctl->tmem_base;

  // unit of this CTA's pair within quad unit `tu`: pair 0 -> (m_blk, n_blk), pair 1 -> (width, flags)
#define DMUON_QUAD_UNIT(tu, mu, nu, share_a, share_b)                      \
  const int mu = pair ? (tu).width : (tu).m_blk;                          \
  const int nu = pair ? (tu).flags : (tu).n_blk;                          \
  const bool share_a = (tu).m_blk == (tu).width;                          \
  const bool share_b = (tu).n_blk == (tu).flags;

  if (warp == 0) {
    // ================================================================== TMA producer (all four CTAs)
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      const uint16_t mc_mask = static_cast<uint16_t>((1u << half) | (1u << (half + 2)));   // same half of both pairs
      for (int u = worker; u < total_units; u += num_workers) {
        const int p = u / units_per_problem;
        const TileUnit tu = units[u - p * units_per_problem];
        const GemmProblem* pr = probs + p;
        const uint64_t tmA = reinterpret_cast<uint64_t>(&pr->tmA);
        const uint64_t tmB = reinterpret_cast<uint64_t>(&pr->tmB);
        const int un = u + num_workers;
        if (un < total_units) {
          const int pn = un / units_per_problem;
          if (pn != p) {
            tma_prefetch_desc(reinterpret_cast<uint64_t>(&probs[pn].tmA));
            tma_prefetch_desc(reinterpret_cast<uint64_t>(&probs[pn].tmB));
          }
        }
        DMUON_QUAD_UNIT(tu, mu, nu, share_a, share_b)
        const int a_blk = 2 * mu + static_cast<int>(half);
        const int b_blk = 2 * nu + static_cast<int>(half);
        for (int kb = 0; kb < k_blocks; ++kb) {
          mbar_wait(bar_empty + 8 * stage, phase ^ 1);
          const uint32_t sA = base + stage * kStageBytes;
          const uint32_t sB = sA + kBlockBytes;
          if (half == 0) mbar_expect_tx(bar_full + 8 * stage, 2 * kStageBytes);   // both CTAs' halves of the stage
          const uint32_t fb = mapa(bar_full + 8 * stage, leader);                  // unicast: the leader's barrier
          const uint32_t fm = bar_full + 8 * stage;                                // multicast: each pair's leader
          if (!share_a) tma_load_2d_pair(sA, tmA, kb * kBlkK, a_blk * kBlk, fb);
          else if (pair == 0) tma_load_2d_pair_mcast(sA, tmA, kb * kBlkK, a_blk * kBlk, fm, mc_mask);
          if (!kBMn) {
            if (!share_b) tma_load_2d_pair(sB, tmB, kb * kBlkK, b_blk * kBlk, fb);
            else if (pair == 0) tma_load_2d_pair_mcast(sB, tmB, kb * kBlkK, b_blk * kBlk, fm, mc_mask);
          } else {
            if (!share_b) {
              tma_load_2d_pair(sB, tmB, b_blk * kBlk, kb * kBlkK, fb);
              tma_load_2d_pair(sB + kBlockBytes / 2, tmB, b_blk * kBlk + 64, kb * kBlkK, fb);
            } else if (pair == 0) {
              tma_load_2d_pair_mcast(sB, tmB, b_blk * kBlk, kb * kBlkK, fm, mc_mask);
              tma_load_2d_pair_mcast(sB + kBlockBytes / 2, tmB, b_blk * kBlk + 64, kb * kBlkK, fm, mc_mask);
            }
          }
          if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
      }
    }
    __syncwarp();
  } else if (warp == 1) {
    // ================================================================== MMA issuer (leader CTA of each pair)
    if (lane == 0 && half == 0) {
      int stage = 0;
      uint32_t phase = 0;
      int it = 0;
      const uint32_t idesc = make_idesc(256, 256, kBMn);
      for (int u = worker; u < total_units; u += num_workers, ++it) {
        const int as = it & 1;
        const uint32_t aphase = (it >> 1) & 1;
        mbar_wait(bar_tempty + 8 * as, aphase ^ 1);
        tcgen05_fence_after();
        const uint32_t d_tmem = tmem_base + as * kAccCols;
        for (int kb = 0; kb < k_blocks; ++kb) {
          mbar_wait(bar_full + 8 * stage, phase);
          tcgen05_fence_after();
          const uint32_t sA = base + stage * kStageBytes;
          const uint32_t sB = sA + kBlockBytes;
#pragma unroll
          for (int k = 0; k < kBlkK / 16; ++k) {
            const uint64_t ad = desc_kmajor(sA + k * 32);
            const uint64_t bd = kBMn ? desc_mnmajor(sB + k * 2048) : desc_kmajor(sB + k * 32);
            mma_f16<2>(d_tmem, ad, bd, idesc, (kb | k) != 0);
          }
          mma_commit_pair(bar_empty + 8 * stage, 0xF);           // slot consumed by this pair: tell all four CTAs
          if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
        mma_commit_pair(bar_tfull + 8 * as, pair_mask);
      }
    }
    __syncwarp();
  } else {
    // ================================================================== epilogue (warps 2..5)
    const int q = warp & 3;
    const int row = q * 32 + lane;
    const uint32_t tempty_leader = mapa(bar_tempty, leader);
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
      DMUON_QUAD_UNIT(tu, mu, nu, share_a, share_b)
      const bool duplicate = share_a && share_b && pair == 1;     // odd leftover: pair 1 shadows pair 0, stores nothing
      const int bi = 2 * mu + static_cast<int>(half);
      const int bj0 = 2 * nu;
      const int64_t grow = static_cast<int64_t>(bi) * kBlk + row;
      const int64_t gcol0 = static_cast<int64_t>(bj0) * kBlk;
      int c_lo = 0, c_hi = 0;
      if (bi < mb && !duplicate) {
        c_lo = (kSym && bi > bj0) ? (bi - bj0) * 4 : 0;
        c_hi = (nb - bj0 < 2 ? nb - bj0 : 2) * 4;
      }
      Addends a0 = {}, a1 = {};
      if (c_lo < c_hi) load_addends<kOp>(a0, D, D2, ldc, grow, gcol0 + c_lo * 32);
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
      tcgen05_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster(tempty_leader + 8 * as);
    }
  }
#undef DMUON_QUAD_UNIT

  tcgen05_fence_before();
  cluster_sync();
  if (warp == 1) tmem_dealloc<2>(tmem_base, kTmemCols);
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

#define DMUON_QUAD_ENTRY(name, op)                                                                              \
  __global__ void __launch_bounds__(kQuadThreads, 1)                                                            \
  name(const GemmProblem* __restrict__ probs, const TileUnit* __restrict__ units, int units_per_problem,       \
       int total_units, int k_blocks, int mb, int nb, float alpha, float beta, float beta2) {                   \
    ns_gemm_quad_body<op>(probs, units, units_per_problem, total_units, k_blocks, mb, nb, alpha, beta, beta2);  \
  }
DMUON_QUAD_ENTRY(ns_syrk_xxt_quad_kernel, OP_SYRK)
DMUON_QUAD_ENTRY(ns_sq_poly_quad_kernel, OP_SQ)
DMUON_QUAD_ENTRY(ns_bx_update_quad_kernel, OP_BX)
DMUON_QUAD_ENTRY(ns_gram_acc_quad_kernel, OP_SQ2)
#undef DMUON_QUAD_ENTRY

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

// Quad launch: clusters of 4; as many clusters as can be co-resident (GPC boundaries may leave a few SMs unused).
int launch_quad(GemmKernel kern, int slot, const GemmLaunch& L, cudaStream_t stream) {
  static bool configured[kNumOps] = {};
  static int max_clusters[kNumOps] = {};
  constexpr int kSmem = smem_bytes<true>();
  const int total = L.units_per_problem * L.num_problems;
  if (total <= 0) return DMUON_OK;
  cudaLaunchConfig_t cfg = {};
  cfg.blockDim = dim3(kQuadThreads);
  cfg.dynamicSmemBytes = kSmem;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = 4;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  if (!configured[slot]) {
    DMUON_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmem));
    cfg.gridDim = dim3(4 * (L.grid / 4));
    int n = 0;
    DMUON_CUDA_CHECK(cudaOccupancyMaxActiveClusters(&n, kern, &cfg));
    if (n < 1) { set_error("launch_quad: no cluster of 4 CTAs fits"); return DMUON_ERR_CUDA; }
    max_clusters[slot] = n < L.grid / 4 ? n : L.grid / 4;
    configured[slot] = true;
    if (getenv("DMUON_LOG")) fprintf(stderr, "[dmuon] quad tiling op %d: %d co-resident clusters of 4 (occupancy query %d, %d SMs)\n", slot, max_clusters[slot], n, L.grid);
  }
  const int use = max_clusters[slot] < total ? max_clusters[slot] : total;
  cfg.gridDim = dim3(4 * use);
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
  static const GemmKernel kQuadK[kNumOps] = {ns_syrk_xxt_quad_kernel, ns_sq_poly_quad_kernel, ns_bx_update_quad_kernel,
                                             ns_gram_acc_quad_kernel};
  if (L.quad) return launch_quad(kQuadK[L.op], L.op, L, stream);
  if (L.pair) return launch_op<true>(kPairK[L.op], &configured[kNumOps + L.op], L, stream);
  return launch_op<false>(kSingle[L.op], &configured[L.op], L, stream);
}

}  // namespace dmuon
