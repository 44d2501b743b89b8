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
// Three tilings of one warp-specialised pipeline (warp 0 = TMA producer, warp 1 = tcgen05.mma issuer and TMEM owner,
// then the epilogue warps: TMEM -> registers -> shared-memory tile -> bulk tensor store):
//
//   single CTA  (cta_group::1)  one CTA per SM computes a 128 x 128 or 128 x 256 unit; 3-stage ring of 48 KB.
//   CTA pair    (cta_group::2)  a cluster of two CTAs (one TPC) computes a 256 x 256 unit with UMMA M = 256, N = 256:
//                               each CTA stages its 128 rows of operand A and its 128 columns of operand B (32 KB per
//                               stage, 5 stages) and holds its 128 accumulator rows in its own TMEM, so a unit moves
//                               2/3 of the L2->SMEM bytes per FLOP of the single-CTA tiling.  The leader CTA issues the
//                               MMAs; both producers signal the leader's "full" barrier; tcgen05.commit multicasts the
//                               "slot free" and "accumulator ready" arrivals to both CTAs.
//   CTA pair, 8 epilogue warps  two warps per TMEM lane quarter take alternate 32-column chunks (short contractions,
//                               where the epilogue sets the pace); 4 stages.
//
// Operands are fp16, 128-byte-swizzled tiles moved by cp.async.bulk.tensor; accumulators are fp32 in TMEM, two
// of them (2 x 256 columns) so the epilogue of one unit overlaps the mainloop of the next.  The symmetric ops visit
// only upper-triangular blocks and store each off-diagonal 128 x 128 block twice (direct and mirrored), so the dense
// output later steps need is kept.
//
// Two kinds of kernels are built from the same role functions (produce_phase / mma_phase / epilogue_phase): one
// product per launch (ns_*_kernel, any tiling), and the PROGRAM kernel (ns_program_kernel, CTA pair): every product
// of a bucket's NS program in one launch, chained by per-matrix completion counters, the matrices taken in groups
// sized to the L2 (see "program kernel" below).
#include <cstdio>
#include <cstdlib>
#include <cstring>

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
constexpr int kSchedDepth = 4;                  // program kernel: unit indices the scheduler may run ahead of its readers
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
  uint64_t sched_full[kSchedDepth];             // program kernel: unit index of slot s published (own barrier)
  uint64_t sched_empty[kSchedDepth];            // ... and read by every reader of both CTAs (leader's barrier)
  int32_t sched[kSchedDepth];
  uint64_t addend[kMaxEpiWarps][kEpiAddTiles];     // "addend tile(s) of ring slot s have landed", per epilogue warp
  uint32_t tmem_base;
  uint32_t pad;
};
constexpr int kCtlBytes = 640;
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
  int pend;           // program kernel: matrix whose previous unit this warp has stored but not yet announced, or -1
  uint32_t par;       // bit s: parity of the next completion of addend barrier s (the ring depth differs between
                      // products, so in the program kernel the phases of the barriers cannot be derived from `consumed`)
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
    mbar_wait(ep.abar + 8 * s, (ep.par >> s) & 1u);
    ep.par ^= 1u << s;
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
// The pipeline is written as three role functions over one PHASE (= one product over a range of problems), with the
// pipeline state (ring position, accumulator turn, epilogue staging counters) held by the caller, so that the same code
// serves the one-product kernels (one phase per launch) and the program kernel (all products of a bucket in one
// launch, phases chained by per-matrix completion counters instead of kernel boundaries).
struct PhaseArgs {
  const GemmProblem* probs;     // problems of this phase (device)
  const TileUnit* units;
  const MatRec* recs;
  int units_per_problem, total_units, k_blocks, mb, nb;   // mb, nb: extent of the output in 128-blocks; pair units may
                                                           // overhang it (operands zero-filled, stores skipped)
  Scalars sc;
  // program kernel only
  int first;                    // running index of the phase's first unit: worker w takes the units u with (first + u) % W == w
  uint32_t* done;               // per-problem count of finished (unit, epilogue warp) pairs, or null
  uint32_t need;                // value a problem's counter must have reached before its units of this phase may start
};

struct Ctx {
  uint32_t base, epi_addr, ctl_addr, bar_full, bar_empty, bar_tfull, bar_tempty, tmem_base;
  int warp, lane, worker, num_workers;
  uint32_t rank;
};
struct RingState { int stage; uint32_t phase; };

__device__ __forceinline__ uint32_t ld_acquire_gpu(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void red_release_gpu_add(uint32_t* p, uint32_t v) {
  asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
// Program kernel: wait until every unit of the earlier products of this matrix has been stored (by any CTA).  The
// stores were bulk tensor stores (async proxy) completed before the release; the loads that follow are bulk tensor
// loads: a proxy fence on each side.
__device__ __forceinline__ void wait_done(const uint32_t* ctr, uint32_t need) {
  // (the 20 s limit applies in a DMUON_WATCHDOG build only, see umma.cuh)
  if (ld_acquire_gpu(ctr) < need) {
    const uint64_t t0 = global_timer_ns();
    uint32_t polls = 0;
    while (ld_acquire_gpu(ctr) < need) {
      __nanosleep(100);
      if ((++polls & 0x3FFu) == 0 && global_timer_ns() - t0 > 20000000000ull) DMUON_WATCHDOG_TRAP();
    }
  }
  asm volatile("fence.proxy.async;" ::: "memory");
}
// At most n of this thread's most recent bulk groups may still be in flight (n <= 8: chunks of one unit and warp).
__device__ __forceinline__ void bulk_wait_pending(int n) {
  switch (n) {
    case 0: asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); break;
    case 1: asm volatile("cp.async.bulk.wait_group 1;" ::: "memory"); break;
    case 2: asm volatile("cp.async.bulk.wait_group 2;" ::: "memory"); break;
    case 3: asm volatile("cp.async.bulk.wait_group 3;" ::: "memory"); break;
    case 4: asm volatile("cp.async.bulk.wait_group 4;" ::: "memory"); break;
    case 5: asm volatile("cp.async.bulk.wait_group 5;" ::: "memory"); break;
    case 6: asm volatile("cp.async.bulk.wait_group 6;" ::: "memory"); break;
    case 7: asm volatile("cp.async.bulk.wait_group 7;" ::: "memory"); break;
    default: asm volatile("cp.async.bulk.wait_group 8;" ::: "memory"); break;
  }
}
// Program kernel, lane 0 of an epilogue warp: announce the unit stored before the current one.  `newer` = bulk groups
// committed since (those of the current unit, which may still be in flight).
__device__ __forceinline__ void announce_pending(EpiPipe& ep, uint32_t* done, int newer) {
  if (ep.pend < 0) return;
  bulk_wait_pending(newer);
  asm volatile("fence.proxy.async;" ::: "memory");
  red_release_gpu_add(done + ep.pend, 1u);
  ep.pend = -1;
}
__device__ __forceinline__ int first_unit(const Ctx& c, const PhaseArgs& a) {
  const int r = a.first % c.num_workers;
  return c.worker >= r ? c.worker - r : c.worker + c.num_workers - r;
}

// ================================================================== TMA producer (one lane; both CTAs of a pair)
// One unit of a phase; `un` = this worker's next unit of the phase (descriptor prefetch) or a value >= total_units.
template <int kOp, bool kPair, int kEW>
__device__ __forceinline__ void produce_unit(const Ctx& c, const PhaseArgs& a, int u, int un, RingState& rs) {
  constexpr bool kAMn = op_a_mn(kOp);
  constexpr bool kBMn = op_b_mn(kOp);
  constexpr int kStages = Tiling<kPair, kEW>::kStages;
  constexpr int kStageBytes = Tiling<kPair, kEW>::kStageBytes;
  {
    const int p = u / a.units_per_problem;
    const TileUnit tu = a.units[u - p * a.units_per_problem];
    const GemmProblem* pr = a.probs + p;
    const uint64_t tmA = reinterpret_cast<uint64_t>(&pr->tmA);
    const uint64_t tmB = reinterpret_cast<uint64_t>(&pr->tmB);
    // the next unit of this worker usually belongs to another matrix: fetch its descriptors ahead of use
    if (un < a.total_units) {
      const int pn = un / a.units_per_problem;
      if (pn != p) {
        tma_prefetch_desc(reinterpret_cast<uint64_t>(&a.probs[pn].tmA));
        tma_prefetch_desc(reinterpret_cast<uint64_t>(&a.probs[pn].tmB));
      }
    }
    if (a.done && a.need) wait_done(a.done + pr->rec, a.need);
    const int a_blk = kPair ? 2 * tu.m_blk + static_cast<int>(c.rank) : tu.m_blk;      // this CTA's 128 rows of A
    const int b_blk = kPair ? 2 * tu.n_blk + static_cast<int>(c.rank) : tu.n_blk;      // its first 128 columns of B
    const int w = kPair ? 1 : tu.width;
    for (int kb = 0; kb < a.k_blocks; ++kb) {
      mbar_wait(c.bar_empty + 8 * rs.stage, rs.phase ^ 1);
      const uint32_t sA = c.base + rs.stage * kStageBytes;
      const uint32_t sB = sA + kBlockBytes;
      if (!kPair) {
        const uint32_t fb = c.bar_full + 8 * rs.stage;
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
        if (c.rank == 0) mbar_expect_tx(c.bar_full + 8 * rs.stage, 2 * kStageBytes);
        const uint32_t fb = mapa(c.bar_full + 8 * rs.stage, 0);
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
      if (++rs.stage == kStages) { rs.stage = 0; rs.phase ^= 1; }
    }
  }
}
template <int kOp, bool kPair, int kEW>
__device__ __forceinline__ void produce_phase(const Ctx& c, const PhaseArgs& a, RingState& rs) {
  for (int u = first_unit(c, a); u < a.total_units; u += c.num_workers) produce_unit<kOp, kPair, kEW>(c, a, u, u + c.num_workers, rs);
}

// ================================================================== MMA issuer (one lane; leader CTA only in a pair)
template <int kOp, bool kPair, int kEW>
__device__ __forceinline__ void mma_unit(const Ctx& c, const PhaseArgs& a, int u, RingState& rs, int it) {
  constexpr bool kAMn = op_a_mn(kOp);
  constexpr bool kBMn = op_b_mn(kOp);
  constexpr int kCG = kPair ? 2 : 1;
  constexpr int kStages = Tiling<kPair, kEW>::kStages;
  constexpr int kStageBytes = Tiling<kPair, kEW>::kStageBytes;
  {
    const int p = u / a.units_per_problem;
    const TileUnit tu = a.units[u - p * a.units_per_problem];
    const uint32_t idesc = make_idesc(kPair ? 256 : 128, kPair ? 256 : tu.width * kBlk, kAMn, kBMn);
    const int as = it & 1;
    const uint32_t aphase = (it >> 1) & 1;
    mbar_wait(c.bar_tempty + 8 * as, aphase ^ 1);    // epilogue has drained this accumulator
    tcgen05_fence_after();
    const uint32_t d_tmem = c.tmem_base + as * kAccCols;
    for (int kb = 0; kb < a.k_blocks; ++kb) {
      mbar_wait(c.bar_full + 8 * rs.stage, rs.phase);       // TMA bytes have landed (in both CTAs of a pair)
      tcgen05_fence_after();
      const uint32_t sA = c.base + rs.stage * kStageBytes;
      const uint32_t sB = sA + kBlockBytes;
#pragma unroll
      for (int k = 0; k < kBlkK / 16; ++k) {
        const uint64_t ad = kAMn ? desc_mnmajor(sA + k * 2048) : desc_kmajor(sA + k * 32);
        const uint64_t bd = kBMn ? desc_mnmajor(sB + k * 2048) : desc_kmajor(sB + k * 32);
        mma_f16<kCG>(d_tmem, ad, bd, idesc, (kb | k) != 0);
      }
      // frees the smem slot (in both CTAs) when these MMAs finish
      if (kPair) mma_commit_pair(c.bar_empty + 8 * rs.stage, 3); else mma_commit(c.bar_empty + 8 * rs.stage);
      if (++rs.stage == kStages) { rs.stage = 0; rs.phase ^= 1; }
    }
    // accumulator complete -> epilogue (of both CTAs)
    if (kPair) mma_commit_pair(c.bar_tfull + 8 * as, 3); else mma_commit(c.bar_tfull + 8 * as);
  }
}
template <int kOp, bool kPair, int kEW>
__device__ __forceinline__ void mma_phase(const Ctx& c, const PhaseArgs& a, RingState& rs, int& it) {
  for (int u = first_unit(c, a); u < a.total_units; u += c.num_workers, ++it) mma_unit<kOp, kPair, kEW>(c, a, u, rs, it);
}

// ================================================================== epilogue (kEW warps: TMEM lane quarter warp % 4;
//                                                                    with two warps per quarter, alternate chunks)
template <int kOp, bool kPair, int kEpi, int kEW>
__device__ __forceinline__ void epilogue_unit(const Ctx& c, const PhaseArgs& a, int u, EpiPipe& ep, int it) {
  constexpr bool kSym = op_symmetric(kOp);
  constexpr int kSub = EpiCfg<kEW>::kSub;
  constexpr int kRing = op_ring(kOp);
  const int lane = c.lane;
  const int q = c.warp & 3;
  const int sub = (c.warp - 2) >> 2;
  const int row = q * 32 + lane;
  const uint32_t tempty_leader = kPair ? mapa(c.bar_tempty, 0) : c.bar_tempty;
  const Scalars& sc = a.sc;
  ep.issued = ep.consumed = 0;      // every requested addend tile was read by the end of its unit: ring slots restart at 0
  {
    const int p = u / a.units_per_problem;
    const TileUnit tu = a.units[u - p * a.units_per_problem];
    const GemmProblem* pr = a.probs + p;
    EpiCtx x;
    x.tmC = reinterpret_cast<uint64_t>(&pr->tmC);
    x.tmD = reinterpret_cast<uint64_t>(&pr->tmD);
    x.tmD2 = reinterpret_cast<uint64_t>(&pr->tmD2);
    x.fin.ldw = pr->ldc;
    x.fin.W = nullptr;
    x.fin.W32 = nullptr;
    x.fin.so = 0.f;
    if (kEpi != EPI_F16) {
      const MatRec& rec = a.recs[sc.rec_base + pr->rec];
      x.fin.W = static_cast<uint16_t*>(rec.W);
      x.fin.W32 = rec.W32;
      x.fin.so = kEpi == EPI_BF16 ? rec.inv_xscale : sc.lr * rec.scale * rec.inv_xscale;
    }
    const int as = it & 1;
    const uint32_t aphase = (it >> 1) & 1;
    const int bi = kPair ? 2 * tu.m_blk + static_cast<int>(c.rank) : tu.m_blk;      // row block of this CTA
    const int bj0 = kPair ? 2 * tu.n_blk : tu.n_blk;                               // first column block
    const int nbk = kPair ? 2 : tu.width;
    const int64_t grow = static_cast<int64_t>(bi) * kBlk + row;
    const int wrow0 = bi * kBlk + q * 32;                                          // first row of this warp
    const int gcol0 = bj0 * kBlk;
    // chunks (32 columns each) this warp stores: inside the matrix and, for symmetric results, not left of the
    // diagonal block (those blocks are written by the mirror of another unit)
    int c_lo = 0, c_hi = 0;
    if (bi < a.mb) {
      c_lo = (kSym && bi > bj0) ? (bi - bj0) * 4 : 0;
      c_hi = (a.nb - bj0 < nbk ? a.nb - bj0 : nbk) * 4;
    }
    // addend tiles of this warp's first chunks and its first W words: requested before the accumulator is ready
    const int c0 = c_lo + sub;
    if (op_has_addend(kOp) && lane == 0) {
      if (a.done && a.need && c0 < c_hi) {     // the addend is an earlier product's result
        // (never block with an unannounced unit: another CTA's wait may be for it)
        if (ep.pend >= 0 && ld_acquire_gpu(a.done + pr->rec) < a.need) announce_pending(ep, a.done, 0);
        wait_done(a.done + pr->rec, a.need);
      }
      for (int j = 0; j < kRing - 1; ++j)
        if (c0 + j * kSub < c_hi) addend_issue<kOp, kEW>(ep, x, gcol0 + (c0 + j * kSub) * 32, wrow0);
    }
    WWords w0 = {}, w1 = {};
    if (c0 < c_hi) load_w<kEpi>(w0, x.fin, grow, gcol0 + c0 * 32);
    if (a.done && lane == 0 && ep.pend >= 0 && !mbar_try_wait(c.bar_tfull + 8 * as, aphase)) announce_pending(ep, a.done, 0);
    const uint32_t nout0 = ep.nout;
    mbar_wait_warp(c.bar_tfull + 8 * as, aphase, DMUON_EPI_SLEEP_NS);
    tcgen05_fence_after();
    const uint32_t taddr = c.tmem_base + as * kAccCols + (static_cast<uint32_t>(q * 32) << 16);
    for (int cc = c0; cc < c_hi; cc += 2 * kSub) {
      uint32_t v[32];
      const int cn = cc + kSub;
      if (op_has_addend(kOp) && lane == 0 && cc + (kRing - 1) * kSub < c_hi) addend_issue<kOp, kEW>(ep, x, gcol0 + (cc + (kRing - 1) * kSub) * 32, wrow0);
      if (cn < c_hi) load_w<kEpi>(w1, x.fin, grow, gcol0 + cn * 32);
      tmem_ld_32x32(taddr + cc * 32, v);
      tmem_wait_ld();
      epilogue_chunk<kOp, kEpi, kEW>(v, w0, x, ep, grow, gcol0 + cc * 32, sc, bj0 + (cc >> 2) != bi);
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
      if (kPair) mbar_arrive_cluster(tempty_leader + 8 * as); else mbar_arrive(c.bar_tempty + 8 * as);
      if (a.done) {
        // program kernel: once this warp's part of a unit is in global memory the matrix's later products may read it.
        // Announced one unit late (its bulk stores have completed by then, nothing stalls), or earlier whenever this
        // warp would otherwise block (above) and at the end of the phase.
        announce_pending(ep, a.done, static_cast<int>(ep.nout - nout0));
        ep.pend = pr->rec;
      }
    }
  }
}
template <int kOp, bool kPair, int kEpi, int kEW>
__device__ __forceinline__ void epilogue_phase(const Ctx& c, const PhaseArgs& a, EpiPipe& ep, int& it) {
  for (int u = first_unit(c, a); u < a.total_units; u += c.num_workers, ++it) epilogue_unit<kOp, kPair, kEpi, kEW>(c, a, u, ep, it);
  if (a.done && c.lane == 0) announce_pending(ep, a.done, 0);
}

template <bool kPair, int kEW>
__device__ __forceinline__ Ctx pipeline_setup() {
  constexpr int kCG = kPair ? 2 : 1;
  constexpr int kStages = Tiling<kPair, kEW>::kStages;
  constexpr int kStageBytes = Tiling<kPair, kEW>::kStageBytes;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  Ctx c;
  c.base = (raw + 1023u) & ~1023u;    // swizzle-128B atoms need 1024-byte alignment
  // [operand ring | epilogue tiles (2 KB each, 1024-byte aligned) | barriers]
  c.epi_addr = c.base + kStages * kStageBytes;
  c.ctl_addr = c.epi_addr + EpiCfg<kEW>::kBytes;
  SmemCtl* ctl = reinterpret_cast<SmemCtl*>(smem_raw + (c.ctl_addr - raw));
  c.bar_full = c.ctl_addr + offsetof(SmemCtl, full);
  c.bar_empty = c.ctl_addr + offsetof(SmemCtl, empty);
  c.bar_tfull = c.ctl_addr + offsetof(SmemCtl, tmem_full);
  c.bar_tempty = c.ctl_addr + offsetof(SmemCtl, tmem_empty);
  c.warp = threadIdx.x >> 5;
  c.lane = threadIdx.x & 31;
  c.rank = kPair ? cluster_ctarank() : 0u;          // 0 = leader of the pair
  c.worker = kPair ? (blockIdx.x >> 1) : blockIdx.x;
  c.num_workers = kPair ? (gridDim.x >> 1) : gridDim.x;
  if (threadIdx.x == 0) {
    for (int s = 0; s < kStages; ++s) {
      mbar_init(c.bar_full + 8 * s, 1);
      mbar_init(c.bar_empty + 8 * s, 1);
    }
    for (int s = 0; s < 2; ++s) {
      mbar_init(c.bar_tfull + 8 * s, 1);
      mbar_init(c.bar_tempty + 8 * s, kPair ? 2 * kEW : kEW);   // one arrival per epilogue warp (of both CTAs)
    }
    for (int s = 0; s < kEW * kEpiAddTiles; ++s) mbar_init(c.ctl_addr + offsetof(SmemCtl, addend) + 8 * s, 1);
    for (int s = 0; s < kSchedDepth; ++s) {
      mbar_init(c.ctl_addr + offsetof(SmemCtl, sched_full) + 8 * s, 1);
      // readers: the leader's MMA thread and epilogue warps, the peer's producer and epilogue warps
      mbar_init(c.ctl_addr + offsetof(SmemCtl, sched_empty) + 8 * s, kPair ? 2 + 2 * kEW : 1 + kEW);
    }
    fence_barrier_init();
  }
  if (c.warp == 1) tmem_alloc<kCG>(c.ctl_addr + offsetof(SmemCtl, tmem_base), kTmemCols);
  tcgen05_fence_before();
  if (kPair) cluster_sync(); else __syncthreads();
  tcgen05_fence_after();
  c.tmem_base = ctl->tmem_base;
  return c;
}
template <bool kPair, int kEW>
__device__ __forceinline__ EpiPipe epilogue_pipe(const Ctx& c) {
  EpiPipe ep;
  ep.obuf = c.epi_addr + (c.warp - 2) * EpiCfg<kEW>::kWarpBytes;
  ep.abar = c.ctl_addr + offsetof(SmemCtl, addend) + (c.warp - 2) * (8 * kEpiAddTiles);
  ep.issued = ep.consumed = ep.nout = 0;
  ep.par = 0;
  ep.pend = -1;
  return ep;
}
template <bool kPair>
__device__ __forceinline__ void pipeline_teardown(const Ctx& c) {
  tcgen05_fence_before();
  if (kPair) cluster_sync(); else __syncthreads();
  if (c.warp == 1) tmem_dealloc<kPair ? 2 : 1>(c.tmem_base, kTmemCols);
}

// One product per launch.
template <int kOp, bool kPair, int kEpi, int kEW>
__device__ __forceinline__ void ns_gemm_body(const GemmProblem* __restrict__ probs, const TileUnit* __restrict__ units,
                                             const MatRec* __restrict__ recs, int units_per_problem, int total_units,
                                             int k_blocks, int mb, int nb, const Scalars sc) {
  const Ctx c = pipeline_setup<kPair, kEW>();
  PhaseArgs a;
  a.probs = probs; a.units = units; a.recs = recs;
  a.units_per_problem = units_per_problem; a.total_units = total_units;
  a.k_blocks = k_blocks; a.mb = mb; a.nb = nb;
  a.sc = sc;
  a.first = 0; a.done = nullptr; a.need = 0;
  if (c.warp == 0) {
    if (c.lane == 0) {
      RingState rs{0, 0};
      produce_phase<kOp, kPair, kEW>(c, a, rs);
    }
    __syncwarp();
  } else if (c.warp == 1) {
    if (c.lane == 0 && c.rank == 0) {
      RingState rs{0, 0};
      int it = 0;
      mma_phase<kOp, kPair, kEW>(c, a, rs, it);
    }
    __syncwarp();
  } else {
    EpiPipe ep = epilogue_pipe<kPair, kEW>(c);
    int it = 0;
    epilogue_phase<kOp, kPair, kEpi, kEW>(c, a, ep, it);
    // the bulk stores of this warp must have completed (not only read their tiles) before the CTA exits
    if (c.lane == 0) bulk_wait_all();
    __syncwarp();
  }
  pipeline_teardown<kPair>(c);
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

// ------------------------------------------------------------------------------------------------ program kernel
// ALL products of a bucket's NS program in ONE launch ("grouped by shape and advanced together").  The
// launch has one list of work units -- for each group of matrices, for each product of the program, the units of that
// product over the group -- and the CTA pairs take its entries in order from a global counter.  A unit of product l of
// a matrix starts when every unit of product l - 1 of THAT matrix has been stored (per-matrix counters in global
// memory, bumped by the epilogue warps after their bulk stores completed); nothing else orders the products, so the
// pipeline never drains between them, there is no launch gap, and a group sized to the L2 keeps its G, B, T, R in
// cache from one product to the next -- which is what pays: fewer DRAM bytes, more clock under the power cap.
// CTA-pair tiling, 4 epilogue warps.  Deadlock-free: units are handed to RUNNING CTAs in list order and a unit only
// waits for units earlier in the list.
constexpr int kProgKindGram = 0, kProgKindSq = 1, kProgKindSq2 = 2, kProgKindX = 3, kProgKindXFinal = 4;
struct ProgPhase {
  const GemmProblem* probs;
  float alpha, beta, beta2;
  uint32_t need;            // completions (units x 8 epilogue warps) of a matrix before this product may read its inputs
  int kind;
  int pad;
};
struct alignas(16) ProgParams {
  ProgPhase ph[kMaxProgPhases];
  const TileUnit* units[3];
  const MatRec* recs;
  uint32_t* done;
  uint32_t* queue;          // next unit of the launch's list (dynamic assignment)
  int upp[3];
  int total_units;
  int num_phases, count, group, rec_base;
  int m_blocks, n_blocks;   // oriented shape in 128-blocks (m <= n)
  float lr, lrwd;
  int store_c;
};

// Where unit g of the launch's list lies: group of matrices, product, index inside the product's units of the group.
struct Cursor { int g0, li, base, tot; };
__device__ __forceinline__ int phase_tiling(int kind) { return kind == kProgKindGram ? 0 : (kind >= kProgKindX ? 2 : 1); }
__device__ __forceinline__ int phase_units(const ProgParams& P, int g0, int li) {
  const int gn = P.count - g0 < P.group ? P.count - g0 : P.group;
  return gn * P.upp[phase_tiling(P.ph[li].kind)];
}
__device__ __forceinline__ void locate(const ProgParams& P, Cursor& cur, int g) {     // g never decreases
  while (g >= cur.base + cur.tot) {
    cur.base += cur.tot;
    if (++cur.li == P.num_phases) { cur.li = 0; cur.g0 += P.group; }
    cur.tot = phase_units(P, cur.g0, cur.li);
  }
}
template <bool kTall>
__device__ __forceinline__ PhaseArgs phase_args(const ProgParams& P, const Cursor& cur) {
  const ProgPhase& ph = P.ph[cur.li];
  const int t = phase_tiling(ph.kind);
  PhaseArgs a;
  a.probs = ph.probs + cur.g0;
  a.units = P.units[t];
  a.recs = P.recs;
  a.units_per_problem = P.upp[t];
  a.total_units = cur.tot;
  a.k_blocks = (t == 0 ? P.n_blocks : P.m_blocks) * (kBlk / kBlkK);
  a.mb = (t == 2 && kTall) ? P.n_blocks : P.m_blocks;
  a.nb = (t == 2 && !kTall) ? P.n_blocks : P.m_blocks;
  a.sc = Scalars{ph.alpha, ph.beta, ph.beta2, P.lr, P.lrwd, ph.kind == kProgKindXFinal ? P.store_c : 1, P.rec_base};
  a.first = 0;
  a.done = P.done;
  a.need = ph.need;
  return a;
}

// Dynamic unit assignment: the leader's producer thread takes the next index of the launch's list from a global
// counter and publishes it to every role of both CTAs through a small ring in shared memory.  Units are handed out in
// list order to CTAs that are RUNNING, and a unit waits only for units earlier in the list, so the walk cannot
// deadlock even when other kernels keep some of this grid's CTAs from becoming resident (with a fixed assignment the
// resident CTAs would wait for units of CTAs that never start).
struct SchedReader { uint32_t n; uint32_t full, empty_leader, data; };
template <bool kClusterAcquire>
__device__ __forceinline__ int sched_read(SchedReader& r, bool arrive) {
  const uint32_t s = r.n % kSchedDepth;
  if (kClusterAcquire) mbar_wait_cluster(r.full + 8 * s, (r.n / kSchedDepth) & 1);
  else mbar_wait(r.full + 8 * s, (r.n / kSchedDepth) & 1);
  int g;
  asm volatile("ld.shared.s32 %0, [%1];" : "=r"(g) : "r"(r.data + 4 * s) : "memory");
  if (arrive) mbar_arrive_cluster(r.empty_leader + 8 * s);
  ++r.n;
  return g;
}

template <bool kTall, int kFinalEpi>
__global__ void __launch_bounds__(EpiCfg<4>::kThreads, 1) ns_program_kernel(const __grid_constant__ ProgParams P) {
  constexpr int kGram = kTall ? OP_SYRK_T : OP_SYRK;
  constexpr int kX = kTall ? OP_XB : OP_BX;
  const Ctx c = pipeline_setup<true, 4>();
  const uint32_t bar_sfull = c.ctl_addr + offsetof(SmemCtl, sched_full);
  const uint32_t bar_sempty = c.ctl_addr + offsetof(SmemCtl, sched_empty);
  const uint32_t sdata = c.ctl_addr + offsetof(SmemCtl, sched);
  Cursor cur{0, 0, 0, phase_units(P, 0, 0)};
  SchedReader rd{0u, bar_sfull, mapa(bar_sempty, 0), sdata};
  if (c.warp == 0) {
    if (c.lane == 0) {
      RingState rs{0, 0};
      const uint32_t peer_full = mapa(bar_sfull, 1), peer_data = mapa(sdata, 1);
      auto produce = [&](int g) {
        locate(P, cur, g);
        const PhaseArgs a = phase_args<kTall>(P, cur);
        const int u = g - cur.base;
        switch (P.ph[cur.li].kind) {
          case kProgKindGram: produce_unit<kGram, true, 4>(c, a, u, a.total_units, rs); break;
          case kProgKindSq: produce_unit<OP_SQ, true, 4>(c, a, u, a.total_units, rs); break;
          case kProgKindSq2: produce_unit<OP_SQ2, true, 4>(c, a, u, a.total_units, rs); break;
          default: produce_unit<kX, true, 4>(c, a, u, a.total_units, rs); break;
        }
      };
      if (c.rank == 0) {
        // scheduler: takes the next unit of the list for this CTA pair and publishes it to every role of both CTAs
        uint32_t n = 0;
        auto publish = [&](int g) {
          const uint32_t s = n % kSchedDepth;
          mbar_wait(bar_sempty + 8 * s, ((n / kSchedDepth) & 1) ^ 1);
          asm volatile("st.shared.s32 [%0], %1;" ::"r"(sdata + 4 * s), "r"(g) : "memory");
          asm volatile("st.shared::cluster.s32 [%0], %1;" ::"r"(peer_data + 4 * s), "r"(g) : "memory");
          mbar_arrive(bar_sfull + 8 * s);
          mbar_arrive_cluster(peer_full + 8 * s);
          ++n;
        };
        const uint32_t total = static_cast<uint32_t>(P.total_units);
        uint32_t got = atomicAdd(P.queue, 1u);
        int g = got < total ? static_cast<int>(got) : -1;
        publish(g);
        while (g >= 0) {
          // the next index is requested before this unit's loads go out and used after them: the round trip of the
          // atomic (~1 us) is off the producer's critical path
          got = atomicAdd(P.queue, 1u);
          produce(g);
          g = got < total ? static_cast<int>(got) : -1;
          publish(g);
          if (g >= 0) {
            // descriptors of the next unit's problem, ahead of its first load
            Cursor nx = cur;
            locate(P, nx, g);
            const int t = phase_tiling(P.ph[nx.li].kind);
            const GemmProblem* pr = P.ph[nx.li].probs + nx.g0 + (g - nx.base) / P.upp[t];
            tma_prefetch_desc(reinterpret_cast<uint64_t>(&pr->tmA));
            tma_prefetch_desc(reinterpret_cast<uint64_t>(&pr->tmB));
          }
        }
      } else {
        while (true) {
          const int g = sched_read<true>(rd, true);
          if (g < 0) break;
          produce(g);
        }
      }
    }
    __syncwarp();
  } else if (c.warp == 1) {
    if (c.lane == 0 && c.rank == 0) {
      RingState rs{0, 0};
      for (int it = 0;; ++it) {
        const int g = sched_read<false>(rd, true);
        if (g < 0) break;
        locate(P, cur, g);
        const PhaseArgs a = phase_args<kTall>(P, cur);
        const int u = g - cur.base;
        switch (P.ph[cur.li].kind) {
          case kProgKindGram: mma_unit<kGram, true, 4>(c, a, u, rs, it); break;
          case kProgKindSq: mma_unit<OP_SQ, true, 4>(c, a, u, rs, it); break;
          case kProgKindSq2: mma_unit<OP_SQ2, true, 4>(c, a, u, rs, it); break;
          default: mma_unit<kX, true, 4>(c, a, u, rs, it); break;
        }
      }
    }
    __syncwarp();
  } else {
    EpiPipe ep = epilogue_pipe<true, 4>(c);
    for (int it = 0;; ++it) {
      // (never block with an unannounced unit)
      if (c.lane == 0 && ep.pend >= 0 && !mbar_try_wait(rd.full + 8 * (rd.n % kSchedDepth), (rd.n / kSchedDepth) & 1))
        announce_pending(ep, P.done, 0);
      const int g = c.rank == 0 ? sched_read<false>(rd, false) : sched_read<true>(rd, false);
      __syncwarp();                                   // every lane has read the slot
      if (c.lane == 0) mbar_arrive_cluster(rd.empty_leader + 8 * ((rd.n - 1) % kSchedDepth));
      if (g < 0) break;
      locate(P, cur, g);
      const PhaseArgs a = phase_args<kTall>(P, cur);
      const int u = g - cur.base;
      switch (P.ph[cur.li].kind) {
        case kProgKindGram: epilogue_unit<kGram, true, EPI_F16, 4>(c, a, u, ep, it); break;
        case kProgKindSq: epilogue_unit<OP_SQ, true, EPI_F16, 4>(c, a, u, ep, it); break;
        case kProgKindSq2: epilogue_unit<OP_SQ2, true, EPI_F16, 4>(c, a, u, ep, it); break;
        case kProgKindX: epilogue_unit<kX, true, EPI_F16, 4>(c, a, u, ep, it); break;
        default: epilogue_unit<kX, true, kFinalEpi, 4>(c, a, u, ep, it); break;
      }
    }
    if (c.lane == 0) {
      announce_pending(ep, P.done, 0);
      bulk_wait_all();
    }
    __syncwarp();
  }
  pipeline_teardown<true>(c);
}

typedef void (*ProgKernel)(const ProgParams);
ProgKernel g_prog[2][kNumEpi] = {
    {ns_program_kernel<false, EPI_F16>, ns_program_kernel<false, EPI_BF16>, ns_program_kernel<false, EPI_APPLY>, ns_program_kernel<false, EPI_APPLY_MASTER>},
    {ns_program_kernel<true, EPI_F16>, ns_program_kernel<true, EPI_BF16>, ns_program_kernel<true, EPI_APPLY>, ns_program_kernel<true, EPI_APPLY_MASTER>}};
bool g_prog_configured[2][kNumEpi][kMaxDevices];

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

int launch_ns_program(const ProgLaunch& L, cudaStream_t stream) {
  if (L.num_phases < 1 || L.num_phases > kMaxProgPhases || L.final_epi < 0 || L.final_epi >= kNumEpi || L.group < 1) {
    set_error("launch_ns_program: bad phase count %d / epilogue %d / group %d", L.num_phases, static_cast<int>(L.final_epi), L.group);
    return DMUON_ERR_INVALID_ARG;
  }
  if (L.count <= 0) return DMUON_OK;
  int dev = 0;
  DMUON_CUDA_CHECK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) { set_error("launch_ns_program: device ordinal %d is not supported", dev); return DMUON_ERR_UNSUPPORTED_DEVICE; }
  ProgKernel kern = g_prog[L.tall ? 1 : 0][L.final_epi];
  constexpr int kSmem = smem_bytes<true, 4>();
  if (!g_prog_configured[L.tall ? 1 : 0][L.final_epi][dev]) {
    DMUON_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmem));
    g_prog_configured[L.tall ? 1 : 0][L.final_epi][dev] = true;
  }
  ProgParams P;
  memset(&P, 0, sizeof P);
  uint32_t units_before = 0;
  for (int li = 0; li < L.num_phases; ++li) {
    const ProgPhaseHost& h = L.ph[li];
    ProgPhase& ph = P.ph[li];
    ph.probs = h.probs;
    ph.alpha = h.alpha; ph.beta = h.beta; ph.beta2 = h.beta2;
    const bool last = li + 1 == L.num_phases;
    int t;
    switch (h.op) {
      case OP_SYRK: case OP_SYRK_T: ph.kind = kProgKindGram; t = 0; break;
      case OP_SQ: ph.kind = kProgKindSq; t = 1; break;
      case OP_SQ2: ph.kind = kProgKindSq2; t = 1; break;
      default: ph.kind = last ? kProgKindXFinal : kProgKindX; t = 2; break;
    }
    ph.need = units_before * 8u;       // 2 CTAs x 4 epilogue warps signal each unit
    units_before += static_cast<uint32_t>(L.upp[t]);
  }
  for (int t = 0; t < 3; ++t) { P.units[t] = L.units[t]; P.upp[t] = L.upp[t]; }
  P.recs = L.recs;
  P.done = L.done;
  P.queue = L.done + L.count;
  {
    long total = 0;
    for (int li = 0; li < L.num_phases; ++li) total += L.upp[P.ph[li].kind == kProgKindGram ? 0 : (P.ph[li].kind >= kProgKindX ? 2 : 1)];
    total *= L.count;
    if (total > 0x7fffff00L) { set_error("launch_ns_program: %ld work units", total); return DMUON_ERR_INVALID_ARG; }
    P.total_units = static_cast<int>(total);
  }
  P.num_phases = L.num_phases;
  P.count = L.count;
  P.group = L.group;
  P.rec_base = L.rec_base;
  P.m_blocks = L.m_blocks;
  P.n_blocks = L.n_blocks;
  P.lr = L.lr;
  P.lrwd = L.lrwd;
  P.store_c = L.store_c ? 1 : 0;
  DMUON_CUDA_CHECK(cudaMemsetAsync(L.done, 0, sizeof(uint32_t) * (L.count + 1), stream));   // counters + the unit queue
  const int max_units = L.group * (L.upp[0] > L.upp[2] ? L.upp[0] : L.upp[2]);
  const int workers = L.grid / 2 < max_units ? L.grid / 2 : max_units;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(2 * workers);
  cfg.blockDim = dim3(EpiCfg<4>::kThreads);
  cfg.dynamicSmemBytes = kSmem;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = 2;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  DMUON_CUDA_CHECK(cudaLaunchKernelEx(&cfg, kern, P));
  return DMUON_OK;
}

}  // namespace dmuon
