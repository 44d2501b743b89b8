// Persistent grouped GEMM family for the Gram-form Newton-Schulz step on sm_100a (steps a3, a4, a5 of DESIGN.md, and
// step a6 fused into the last a5 epilogue):
//
//   OP_SYRK    C = alpha X X^T                  (PAPER.md:170 G = X X^T; symmetric kernel of PAPER.md:182)
//   OP_SYRK_T  C = alpha Y^T Y                  (the same Gram matrix of a tall matrix held as stored, Y = X^T)
//   OP_SQ      C = alpha A B^T + beta D         (the polynomial in the Gram matrix; A A = A A^T)
//   OP_SQ2     C = alpha A B^T + beta D + beta2 D2   (symmetric, two addends: the running product of the
//                                                P_i = a_i I + B_i of a Gram block, Eq. 4)
//   OP_BX      C = alpha R X + beta X           (X_{i+1} = P X_i with the a X term in the epilogue)
//   OP_XB      C = alpha Y R + beta Y           (the same update of a tall matrix held as stored)
//
// Epilogues of the two X updates ("elementwise operations ... fused into the same epilogue"): fp16 store
// of the new X; or, for the LAST update of a call, the Muon update itself W' = W - lr (scale O + wd W) (Eq. 1
// PAPER.md:51) on bf16 weights or on fp32 master weights, or the bf16 NS output of dmuon_ns_batched.
//
// Two tilings of one warp-specialised pipeline (warp 0 = TMA producer, warp 1 = tcgen05.mma issuer and TMEM owner,
// warps 2..5 = epilogue: TMEM -> registers -> shared-memory tile -> global):
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
#include "epilogue.cuh"
#include "umma.cuh"

namespace dmuon {
namespace {

using namespace umma;

constexpr int kBlockBytes = kBlk * kBlkK * 2;   // 16 KB: 128 rows x 128 B of one operand block
constexpr int kMaxEpiWarps = 8;
constexpr int kTmemCols = 512;
constexpr int kAccCols = 256;                   // columns per accumulator stage
constexpr int kMaxStages = 6;
#ifndef DMUON_EPI_SLEEP_NS
#define DMUON_EPI_SLEEP_NS 256                  // back-off of the epilogue warps' accumulator wait (0 = plain polling)
#endif

// Epilogue staging, per epilogue warp: tiles of 32 rows x 32 fp16 (64-byte rows, 16-byte chunks XOR-swizzled by
// (row >> 1) & 3 = CU_TENSOR_MAP_SWIZZLE_64B, conflict-free for row-wise 16-byte accesses and for ldmatrix / stmatrix).
//   kOutBufs output tiles + kOutBufs mirrored tiles (a tile is rewritten kOutBufs chunks after its bulk store was issued)
//   4 addend tiles: a ring the warp's elected lane fills by TMA three chunks ahead (two-addend products: two pairs)
// Epilogue warps, kEW: 4 = one per TMEM lane quarter; 8 = two per quarter taking alternate 32-column chunks.  With
// short contractions the epilogue sets the pace and one warp per scheduler hides none of its own latencies (TMEM load,
// addend wait, shared-memory round trips); the second warp does, at the price of single-buffered output tiles and one
// operand stage less.
constexpr int kEpiTileBytes = 32 * 64;
constexpr int kEpiAddTiles = 4;
template <int kEW> struct EpiCfg {
  static constexpr int kSub = kEW / 4;                                          // warps per lane quarter
  static constexpr int kOutBufs = kEW == 4 ? 2 : 1;
  static constexpr int kWarpBytes = (2 * kOutBufs + kEpiAddTiles) * kEpiTileBytes;   // 16 KB / 12 KB
  static constexpr int kBytes = kEW * kWarpBytes;                               // 64 KB / 96 KB
  static constexpr int kThreads = 64 + 32 * kEW;
};

template <bool kPair, int kEW> struct Tiling;
template <> struct Tiling<false, 4> {           // one CTA: A block + up to two B blocks per stage
  static constexpr int kStages = 3;
  static constexpr int kStageBytes = 3 * kBlockBytes;
};
template <> struct Tiling<true, 4> {            // CTA pair: this CTA's A block + its B block per stage
  static constexpr int kStages = 5;
  static constexpr int kStageBytes = 2 * kBlockBytes;
};
template <> struct Tiling<true, 8> {
  static constexpr int kStages = 4;
  static constexpr int kStageBytes = 2 * kBlockBytes;
};

struct SmemCtl {
  uint64_t full[kMaxStages];
  uint64_t empty[kMaxStages];
  uint64_t tmem_full[2];
  uint64_t tmem_empty[2];
  uint64_t addend[kMaxEpiWarps][kEpiAddTiles];     // "addend tile(s) of ring slot s have landed", per epilogue warp
  uint32_t tmem_base;
  uint32_t pad;
};
constexpr int kCtlBytes = 512;
static_assert(sizeof(SmemCtl) <= kCtlBytes, "SmemCtl");
template <bool kPair, int kEW> constexpr int smem_bytes() {
  return Tiling<kPair, kEW>::kStages * Tiling<kPair, kEW>::kStageBytes + EpiCfg<kEW>::kBytes + kCtlBytes + 1024 /*alignment slack*/;
}
static_assert(smem_bytes<true, 4>() <= 232448 && smem_bytes<false, 4>() <= 232448 && smem_bytes<true, 8>() <= 232448, "shared memory budget");

struct Scalars {
  float alpha, beta, beta2;
  float lr, lrwd;
  int store_c;     // fused epilogues: also store fp16(x) to C
  int rec_base;    // MatRec of problem p = recs[rec_base + probs[p].rec]
};

__host__ __device__ constexpr bool op_symmetric(int op) { return op == OP_SYRK || op == OP_SQ || op == OP_SQ2 || op == OP_SYRK_T; }
__host__ __device__ constexpr bool op_a_mn(int op) { return op == OP_SYRK_T; }
__host__ __device__ constexpr bool op_b_mn(int op) { return op == OP_BX || op == OP_SYRK_T; }
__host__ __device__ constexpr bool op_has_addend(int op) { return op != OP_SYRK && op != OP_SYRK_T; }
__host__ __device__ constexpr int op_addends(int op) { return op == OP_SQ2 ? 2 : (op_has_addend(op) ? 1 : 0); }
// addend ring: entries in flight per warp (each entry = the addend tile(s) of one 32-column chunk)
__host__ __device__ constexpr int op_ring(int op) { return op == OP_SQ2 ? kEpiAddTiles / 2 : kEpiAddTiles; }

// ------------------------------------------------------------------------------------------------ epilogue
// All fp16 traffic of the epilogue moves by TMA: the addend tiles come in through a per-warp ring (issued three chunks
// ahead, so their L2 latency is off the critical path), the result tile and, for symmetric results, its transpose go
// out as bulk tensor stores from shared memory.  What is left for the LSU per chunk and warp is 4 swizzled 16-byte
// shared stores, the 4 + 4 ldmatrix.trans / stmatrix of a mirrored tile and 4 shared loads per addend: with short
// contractions (K <= 1024) the epilogue, not the mainloop, sets the pace, and the LSU (shared-memory crossbar and
// global store path, one per SM) was what bounded it when the tiles went out as st.global (profiles/r2_experiments.md).
// Only the bf16 weights of the fused update (and fp32 masters) still take the register path: ld.global.nc / st.global.

// Per-unit epilogue context (pointers of the unit's problem).
struct EpiCtx {
  uint64_t tmC, tmD, tmD2;   // tensor maps (generic addresses of the CUtensorMap objects in the problem table)
  FinalCtx fin;              // fused epilogues: the caller's tensors of this matrix (ldw = leading dimension of C)
};
// Per-warp staging state; counters run over the whole kernel.
struct EpiPipe {
  uint32_t obuf;      // kOutBufs output tiles, then kOutBufs mirrored tiles, then the addend ring
  uint32_t abar;      // this warp's addend barriers
  uint32_t issued;    // addend ring entries requested so far
  uint32_t consumed;  // ... and read so far
  uint32_t nout;      // chunks stored so far (output tile toggle)
};

// Lane 0: request the addend tile(s) of rows [wrow0, wrow0 + 32), columns [gcol, gcol + 32) into the next ring entry.
template <int kOp, int kEW>
__device__ __forceinline__ void addend_issue(EpiPipe& ep, const EpiCtx& x, int gcol, int wrow0) {
  constexpr int kRing = op_ring(kOp);
  constexpr int kTiles = op_addends(kOp);
  const uint32_t s = ep.issued % kRing;
  const uint32_t bar = ep.abar + 8 * s;
  const uint32_t dst = ep.obuf + 2 * EpiCfg<kEW>::kOutBufs * kEpiTileBytes + s * kTiles * kEpiTileBytes;
  mbar_expect_tx(bar, kTiles * kEpiTileBytes);
  tma_load_2d(dst, x.tmD, gcol, wrow0, bar);
  if (kOp == OP_SQ2) tma_load_2d(dst + kEpiTileBytes, x.tmD2, gcol, wrow0, bar);
  ++ep.issued;
}

// One 32-column chunk of one accumulator row: v = 32 fp32 accumulators of row `grow`, columns [gcol, gcol + 32).
template <int kOp, int kEpi, int kEW>
__device__ __forceinline__ void epilogue_chunk(const uint32_t (&v)[32], const WWords& ww, const EpiCtx& x, EpiPipe& ep,
                                               int64_t grow, int64_t gcol, const Scalars& sc, bool mirror) {
  const int lane = threadIdx.x & 31;
  const int sw = (lane >> 1) & 3;                        // swizzle term of this lane's row
  float r[32];
  if (op_has_addend(kOp)) {
    constexpr int kRing = op_ring(kOp);
    constexpr int kTiles = op_addends(kOp);
    const uint32_t s = ep.consumed % kRing;
    mbar_wait(ep.abar + 8 * s, (ep.consumed / kRing) & 1);
    const uint32_t src = ep.obuf + 2 * EpiCfg<kEW>::kOutBufs * kEpiTileBytes + s * kTiles * kEpiTileBytes + lane * 64;
#pragma unroll
    for (int g = 0; g < 4; ++g) {
      const uint4 d = ld_shared_v4(src + ((g ^ sw) << 4));
      const uint32_t dw[4] = {d.x, d.y, d.z, d.w};
      uint32_t ew[4] = {0u, 0u, 0u, 0u};
      if (kOp == OP_SQ2) {
        const uint4 e = ld_shared_v4(src + kEpiTileBytes + ((g ^ sw) << 4));
        ew[0] = e.x; ew[1] = e.y; ew[2] = e.z; ew[3] = e.w;
      }
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const float2 df = __half22float2(*reinterpret_cast<const __half2*>(&dw[e]));
        float ax = sc.beta * df.x, ay = sc.beta * df.y;
        if (kOp == OP_SQ2) {
          const float2 ef = __half22float2(*reinterpret_cast<const __half2*>(&ew[e]));
          ax = fmaf(sc.beta2, ef.x, ax);
          ay = fmaf(sc.beta2, ef.y, ay);
        }
        r[g * 8 + e * 2] = fmaf(sc.alpha, __uint_as_float(v[g * 8 + e * 2]), ax);
        r[g * 8 + e * 2 + 1] = fmaf(sc.alpha, __uint_as_float(v[g * 8 + e * 2 + 1]), ay);
      }
    }
    ++ep.consumed;
    __syncwarp();                                        // every lane has read the ring slot before lane 0 refills it
  } else {
#pragma unroll
    for (int e = 0; e < 32; ++e) r[e] = sc.alpha * __uint_as_float(v[e]);
  }
  if (kEpi == EPI_F16 || sc.store_c) {
    // fp16 store of the chunk (32 rows x 32 columns per warp) and, for symmetric results, of its mirror image: staged in
    // this warp's shared-memory tiles, sent as bulk tensor stores by lane 0
    uint32_t o[16];
#pragma unroll
    for (int e = 0; e < 16; ++e) o[e] = pack_half2(r[2 * e], r[2 * e + 1]);
    const bool do_mirror = op_symmetric(kOp) && mirror;
    constexpr int kOutBufs = EpiCfg<kEW>::kOutBufs;
    const uint32_t ot = ep.obuf + (ep.nout % kOutBufs) * kEpiTileBytes;
    const uint32_t mt = ot + kOutBufs * kEpiTileBytes;
    // the bulk stores issued from these two tiles kOutBufs chunks ago have read them (one group per chunk)
    if (lane == 0) bulk_wait_read<kOutBufs - 1>();
    __syncwarp();
#pragma unroll
    for (int g = 0; g < 4; ++g) st_shared_v4(ot + lane * 64 + ((g ^ sw) << 4), o[g * 4], o[g * 4 + 1], o[g * 4 + 2], o[g * 4 + 3]);
    if (do_mirror) {
      // transposed tile T[c][r] from the direct tile, 8 x 8 blocks at a time: ldmatrix.trans reads block (rb, cb) of the
      // direct tile transposed into the fragment layout, stmatrix writes it as block (cb, rb) of T
      __syncwarp();
#pragma unroll
      for (int cb = 0; cb < 4; ++cb) {
        uint32_t f0, f1, f2, f3;
        ldmatrix_x4_trans(ot + lane * 64 + ((cb ^ sw) << 4), f0, f1, f2, f3);
        const int trow = 8 * cb + (lane & 7);
        stmatrix_x4(mt + trow * 64 + (((lane >> 3) ^ ((trow >> 1) & 3)) << 4), f0, f1, f2, f3);
      }
    }
    fence_proxy_async();                                 // generic-proxy writes -> visible to the bulk (async-proxy) store
    __syncwarp();
    if (lane == 0) {
      const int wrow0 = static_cast<int>(grow);          // lane 0 holds the warp's first row
      tma_store_2d(x.tmC, ot, static_cast<int>(gcol), wrow0);
      if (do_mirror) tma_store_2d(x.tmC, mt, wrow0, static_cast<int>(gcol));
      bulk_commit();
    }
    ++ep.nout;
  }
  if (kEpi != EPI_F16) final_store<kEpi>(r, ww, x.fin, grow, gcol, sc.lrwd);
}

// ------------------------------------------------------------------------------------------------ the kernel body
// mb, nb: extent of the output in 128-blocks (rows, columns); pair units may overhang it (TMA zero-fills the
// operands there, the epilogue skips those blocks).
template <int kOp, bool kPair, int kEpi, int kEW>
__device__ __forceinline__ void ns_gemm_body(const GemmProblem* __restrict__ probs, const TileUnit* __restrict__ units,
                                             const MatRec* __restrict__ recs, int units_per_problem, int total_units,
                                             int k_blocks, int mb, int nb, const Scalars sc) {
  constexpr bool kSym = op_symmetric(kOp);
  constexpr bool kAMn = op_a_mn(kOp);
  constexpr bool kBMn = op_b_mn(kOp);
  constexpr int kCG = kPair ? 2 : 1;
  constexpr int kStages = Tiling<kPair, kEW>::kStages;
  constexpr int kStageBytes = Tiling<kPair, kEW>::kStageBytes;
  constexpr int kEpiBytes = EpiCfg<kEW>::kBytes;
  constexpr int kEpiWarpBytes = EpiCfg<kEW>::kWarpBytes;
  constexpr int kSub = EpiCfg<kEW>::kSub;

  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;    // swizzle-128B atoms need 1024-byte alignment
  // [operand ring | epilogue tiles (2 KB each, 1024-byte aligned) | barriers]
  const uint32_t epi_addr = base + kStages * kStageBytes;
  const uint32_t ctl_addr = epi_addr + kEpiBytes;
  SmemCtl* ctl = reinterpret_cast<SmemCtl*>(smem_raw + (ctl_addr - raw));
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
      mbar_init(bar_tempty + 8 * s, kPair ? 2 * kEW : kEW);   // one arrival per epilogue warp (of both CTAs)
    }
    for (int s = 0; s < kEW * kEpiAddTiles; ++s) mbar_init(ctl_addr + offsetof(SmemCtl, addend) + 8 * s, 1);
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
            if (!kAMn) {
              tma_load_2d(sA, tmA, kb * kBlkK, a_blk * kBlk, fb);
            } else {
              tma_load_2d(sA, tmA, a_blk * kBlk, kb * kBlkK, fb);                 // 64 (m) x 64 (k) boxes, 8 KB each
              tma_load_2d(sA + kBlockBytes / 2, tmA, a_blk * kBlk + 64, kb * kBlkK, fb);
            }
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
            if (!kAMn) {
              tma_load_2d_pair(sA, tmA, kb * kBlkK, a_blk * kBlk, fb);
            } else {
              tma_load_2d_pair(sA, tmA, a_blk * kBlk, kb * kBlkK, fb);
              tma_load_2d_pair(sA + kBlockBytes / 2, tmA, a_blk * kBlk + 64, kb * kBlkK, fb);
            }
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
        const uint32_t idesc = make_idesc(kPair ? 256 : 128, kPair ? 256 : tu.width * kBlk, kAMn, kBMn);
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
            const uint64_t ad = kAMn ? desc_mnmajor(sA + k * 2048) : desc_kmajor(sA + k * 32);
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
    // ================================================================== epilogue (kEW warps: TMEM lane quarter warp % 4;
    //                                                                    with two warps per quarter, alternate chunks)
    const int q = warp & 3;
    const int sub = (warp - 2) >> 2;
    const int row = q * 32 + lane;
    constexpr int kRing = op_ring(kOp);
    EpiPipe ep;
    ep.obuf = epi_addr + (warp - 2) * kEpiWarpBytes;
    ep.abar = ctl_addr + offsetof(SmemCtl, addend) + (warp - 2) * (8 * kEpiAddTiles);
    ep.issued = ep.consumed = ep.nout = 0;
    const uint32_t tempty_leader = kPair ? mapa(bar_tempty, 0) : bar_tempty;
    int it = 0;
    for (int u = worker; u < total_units; u += num_workers, ++it) {
      const int p = u / units_per_problem;
      const TileUnit tu = units[u - p * units_per_problem];
      const GemmProblem* pr = probs + p;
      EpiCtx x;
      x.tmC = reinterpret_cast<uint64_t>(&pr->tmC);
      x.tmD = reinterpret_cast<uint64_t>(&pr->tmD);
      x.tmD2 = reinterpret_cast<uint64_t>(&pr->tmD2);
      x.fin.ldw = pr->ldc;
      x.fin.W = nullptr;
      x.fin.W32 = nullptr;
      x.fin.so = 0.f;
      if (kEpi != EPI_F16) {
        const MatRec& rec = recs[sc.rec_base + pr->rec];
        x.fin.W = static_cast<uint16_t*>(rec.W);
        x.fin.W32 = rec.W32;
        x.fin.so = kEpi == EPI_BF16 ? rec.inv_xscale : sc.lr * rec.scale * rec.inv_xscale;
      }
      const int as = it & 1;
      const uint32_t aphase = (it >> 1) & 1;
      const int bi = kPair ? 2 * tu.m_blk + static_cast<int>(rank) : tu.m_blk;      // row block of this CTA
      const int bj0 = kPair ? 2 * tu.n_blk : tu.n_blk;                               // first column block
      const int nbk = kPair ? 2 : tu.width;
      const int64_t grow = static_cast<int64_t>(bi) * kBlk + row;
      const int wrow0 = bi * kBlk + q * 32;                                          // first row of this warp
      const int gcol0 = bj0 * kBlk;
      // chunks (32 columns each) this warp stores: inside the matrix and, for symmetric results, not left of the
      // diagonal block (those blocks are written by the mirror of another unit)
      int c_lo = 0, c_hi = 0;
      if (bi < mb) {
        c_lo = (kSym && bi > bj0) ? (bi - bj0) * 4 : 0;
        c_hi = (nb - bj0 < nbk ? nb - bj0 : nbk) * 4;
      }
      // addend tiles of this warp's first chunks and its first W words: requested before the accumulator is ready
      const int c0 = c_lo + sub;
      if (op_has_addend(kOp) && lane == 0) {
        for (int j = 0; j < kRing - 1; ++j)
          if (c0 + j * kSub < c_hi) addend_issue<kOp, kEW>(ep, x, gcol0 + (c0 + j * kSub) * 32, wrow0);
      }
      WWords w0 = {}, w1 = {};
      if (c0 < c_hi) load_w<kEpi>(w0, x.fin, grow, gcol0 + c0 * 32);
      mbar_wait_warp(bar_tfull + 8 * as, aphase, DMUON_EPI_SLEEP_NS);
      tcgen05_fence_after();
      const uint32_t taddr = tmem_base + as * kAccCols + (static_cast<uint32_t>(q * 32) << 16);
      for (int c = c0; c < c_hi; c += 2 * kSub) {
        uint32_t v[32];
        const int cn = c + kSub;
        if (op_has_addend(kOp) && lane == 0 && c + (kRing - 1) * kSub < c_hi) addend_issue<kOp, kEW>(ep, x, gcol0 + (c + (kRing - 1) * kSub) * 32, wrow0);
        if (cn < c_hi) load_w<kEpi>(w1, x.fin, grow, gcol0 + cn * 32);
        tmem_ld_32x32(taddr + c * 32, v);
        tmem_wait_ld();
        epilogue_chunk<kOp, kEpi, kEW>(v, w0, x, ep, grow, gcol0 + c * 32, sc, bj0 + (c >> 2) != bi);
        if (cn < c_hi) {
          if (op_has_addend(kOp) && lane == 0 && cn + (kRing - 1) * kSub < c_hi) addend_issue<kOp, kEW>(ep, x, gcol0 + (cn + (kRing - 1) * kSub) * 32, wrow0);
          if (cn + kSub < c_hi) load_w<kEpi>(w0, x.fin, grow, gcol0 + (cn + kSub) * 32);
          tmem_ld_32x32(taddr + cn * 32, v);
          tmem_wait_ld();
          epilogue_chunk<kOp, kEpi, kEW>(v, w1, x, ep, grow, gcol0 + cn * 32, sc, bj0 + (cn >> 2) != bi);
        }
      }
      // accumulator fully read by this warp: hand it back to the MMA thread
      tcgen05_fence_before();
      __syncwarp();
      if (lane == 0) {
        if (kPair) mbar_arrive_cluster(tempty_leader + 8 * as); else mbar_arrive(bar_tempty + 8 * as);
      }
    }
    // the bulk stores of this warp must have completed (not only read their tiles) before the CTA exits
    if (lane == 0) bulk_wait_all();
    __syncwarp();
  }

  tcgen05_fence_before();
  if (kPair) cluster_sync(); else __syncthreads();
  if (warp == 1) tmem_dealloc<kCG>(tmem_base, kTmemCols);
}

// One named entry point per product, tiling and epilogue, so profiles (ncu -k) and launch lists tell them apart.
#define DMUON_GEMM_ENTRY(name, op, pair, epi, ew)                                                               \
  __global__ void __launch_bounds__(EpiCfg<ew>::kThreads, 1)                                                    \
  name(const GemmProblem* __restrict__ probs, const TileUnit* __restrict__ units,                               \
       const MatRec* __restrict__ recs, int units_per_problem, int total_units, int k_blocks, int mb, int nb,   \
       const Scalars sc) {                                                                                      \
    ns_gemm_body<op, pair, epi, ew>(probs, units, recs, units_per_problem, total_units, k_blocks, mb, nb, sc);  \
  }
// single CTA, CTA pair, CTA pair with 8 epilogue warps
#define DMUON_GEMM_ENTRIES(stem, op, epi)                           \
  DMUON_GEMM_ENTRY(stem##_kernel, op, false, epi, 4)                \
  DMUON_GEMM_ENTRY(stem##_pair_kernel, op, true, epi, 4)            \
  DMUON_GEMM_ENTRY(stem##_pair_ew8_kernel, op, true, epi, 8)
DMUON_GEMM_ENTRIES(ns_syrk_xxt, OP_SYRK, EPI_F16)
DMUON_GEMM_ENTRIES(ns_syrk_xtx, OP_SYRK_T, EPI_F16)
DMUON_GEMM_ENTRIES(ns_sq_poly, OP_SQ, EPI_F16)
DMUON_GEMM_ENTRIES(ns_gram_acc, OP_SQ2, EPI_F16)
DMUON_GEMM_ENTRIES(ns_bx_update, OP_BX, EPI_F16)
DMUON_GEMM_ENTRIES(ns_bx_out, OP_BX, EPI_BF16)
DMUON_GEMM_ENTRIES(ns_bx_apply, OP_BX, EPI_APPLY)
DMUON_GEMM_ENTRIES(ns_bx_apply_master, OP_BX, EPI_APPLY_MASTER)
DMUON_GEMM_ENTRIES(ns_xb_update, OP_XB, EPI_F16)
DMUON_GEMM_ENTRIES(ns_xb_out, OP_XB, EPI_BF16)
DMUON_GEMM_ENTRIES(ns_xb_apply, OP_XB, EPI_APPLY)
DMUON_GEMM_ENTRIES(ns_xb_apply_master, OP_XB, EPI_APPLY_MASTER)
#undef DMUON_GEMM_ENTRIES
#undef DMUON_GEMM_ENTRY

typedef void (*GemmKernel)(const GemmProblem*, const TileUnit*, const MatRec*, int, int, int, int, int, const Scalars);

constexpr int kNumTilings = 3;           // single CTA, CTA pair, CTA pair with 8 epilogue warps
struct KernelEntry {
  GemmKernel fn[kNumTilings];
  bool configured[kNumTilings][kMaxDevices];       // cudaFuncSetAttribute is per device
};
#define DMUON_K(stem) {{stem##_kernel, stem##_pair_kernel, stem##_pair_ew8_kernel}}

// [op][epilogue]; null = combination does not exist (fused epilogues belong to the two X updates)
KernelEntry g_kernels[kNumOps][kNumEpi] = {
    /* OP_SYRK   */ {DMUON_K(ns_syrk_xxt), {}, {}, {}},
    /* OP_SQ     */ {DMUON_K(ns_sq_poly), {}, {}, {}},
    /* OP_BX     */ {DMUON_K(ns_bx_update), DMUON_K(ns_bx_out), DMUON_K(ns_bx_apply), DMUON_K(ns_bx_apply_master)},
    /* OP_SQ2    */ {DMUON_K(ns_gram_acc), {}, {}, {}},
    /* OP_SYRK_T */ {DMUON_K(ns_syrk_xtx), {}, {}, {}},
    /* OP_XB     */ {DMUON_K(ns_xb_update), DMUON_K(ns_xb_out), DMUON_K(ns_xb_apply), DMUON_K(ns_xb_apply_master)},
};
#undef DMUON_K

template <bool kPair, int kEW>
int launch_op(KernelEntry& ke, const GemmLaunch& L, cudaStream_t stream) {
  constexpr int kSmem = smem_bytes<kPair, kEW>();
  constexpr int kTiling = !kPair ? 0 : (kEW == 4 ? 1 : 2);
  GemmKernel kern = ke.fn[kTiling];
  int dev = 0;
  DMUON_CUDA_CHECK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) { set_error("launch_ns_gemm: device ordinal %d is not supported", dev); return DMUON_ERR_UNSUPPORTED_DEVICE; }
  if (!ke.configured[kTiling][dev]) {
    DMUON_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmem));
    ke.configured[kTiling][dev] = true;
  }
  const int total = L.units_per_problem * L.num_problems;
  if (total <= 0) return DMUON_OK;
  const int workers = kPair ? L.grid / 2 : L.grid;
  const int use = workers < total ? workers : total;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(kPair ? 2 * use : use);
  cfg.blockDim = dim3(EpiCfg<kEW>::kThreads);
  cfg.dynamicSmemBytes = kSmem;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = kPair ? 2 : 1;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  Scalars sc{L.alpha, L.beta, L.beta2, L.lr, L.lrwd, L.store_c ? 1 : 0, L.rec_base};
  DMUON_CUDA_CHECK(cudaLaunchKernelEx(&cfg, kern, L.problems, L.units, L.recs, L.units_per_problem, total, L.k_blocks,
                                      L.m_blocks, L.n_blocks, sc));
  return DMUON_OK;
}

}  // namespace

int gemm_smem_bytes() {
  const int a = smem_bytes<false, 4>(), b = smem_bytes<true, 4>(), c = smem_bytes<true, 8>();
  return a > b ? (a > c ? a : c) : (b > c ? b : c);
}

int launch_ns_gemm(const GemmLaunch& L, cudaStream_t stream) {
  if (L.op < 0 || L.op >= kNumOps || L.epi < 0 || L.epi >= kNumEpi) {
    set_error("launch_ns_gemm: bad op %d / epilogue %d", static_cast<int>(L.op), static_cast<int>(L.epi));
    return DMUON_ERR_INVALID_ARG;
  }
  KernelEntry& ke = g_kernels[L.op][L.epi];
  if (!ke.fn[0]) {
    set_error("launch_ns_gemm: op %d has no epilogue %d", static_cast<int>(L.op), static_cast<int>(L.epi));
    return DMUON_ERR_INVALID_ARG;
  }
  if (L.epi != EPI_F16 && !L.recs) { set_error("launch_ns_gemm: fused epilogue without matrix records"); return DMUON_ERR_INVALID_ARG; }
  if (L.pair && L.epi_warps == 8) return launch_op<true, 8>(ke, L, stream);
  if (L.pair) return launch_op<true, 4>(ke, L, stream);
  return launch_op<false, 4>(ke, L, stream);
}

}  // namespace dmuon
