// Persistent grouped GEMM family for the Gram-form Newton-Schulz step on sm_100a (steps a3, a4, a5 of DESIGN.md):
//
//   OP_SYRK  C = alpha * X X^T                (PAPER.md:170 G = X X^T; symmetric kernel of PAPER.md:182)
//   OP_SQ    C = alpha * A A + beta * A       (the polynomial in the Gram matrix; A A = A A^T)
//   OP_BX    C = alpha * B X + beta * X       (X_{i+1} = P X_i with the a X term in the epilogue)
//
// One CTA per SM, warp-specialised:  warp 0 = TMA producer (one thread), warp 1 = tcgen05.mma issuer (one thread)
// and TMEM owner, warps 2..5 = epilogue (TMEM -> registers -> global).  Operands are fp16, staged in a 4-deep
// shared-memory ring of 128-byte-swizzled tiles by cp.async.bulk.tensor; accumulators are fp32 in TMEM, two of
// them (2 x 256 columns) so the epilogue of one work unit overlaps the mainloop of the next.
// The symmetric ops visit only upper-triangular 128 x 128 blocks and store each off-diagonal block twice
// (direct and mirrored), so the dense output later steps need is kept.
#include "common.h"

namespace dmuon {
namespace {

constexpr int kStages = 4;
constexpr int kABytes = kBlk * kBlkK * 2;       // 16 KB: 128 rows x 128 B
constexpr int kBBlockBytes = kBlk * kBlkK * 2;  // 16 KB per 128-wide block of operand B
constexpr int kBBytes = 2 * kBBlockBytes;       // up to two blocks (UMMA N = 256)
constexpr int kStageBytes = kABytes + kBBytes;  // 48 KB
constexpr int kNumThreads = 192;
constexpr int kTmemCols = 512;
constexpr int kAccCols = 256;                   // columns per accumulator stage

struct SmemCtl {
  uint64_t full[kStages];
  uint64_t empty[kStages];
  uint64_t tmem_full[2];
  uint64_t tmem_empty[2];
  uint32_t tmem_base;
  uint32_t pad;
};
constexpr int kSmemBytes = kStages * kStageBytes + 1024 /*alignment slack*/ + 256 /*SmemCtl*/;
static_assert(sizeof(SmemCtl) <= 256, "SmemCtl");

// ------------------------------------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// Spin on the phase parity.  A protocol bug would otherwise hang the GPU, so a (very large) poll bound traps instead.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done = 0;
  uint32_t polls = 0;
  while (true) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(bar), "r"(parity)
        : "memory");
    if (done) break;
    if (++polls > (1u << 28)) __trap();
  }
}

__device__ __forceinline__ void tma_load_2d(uint32_t smem_dst, uint64_t tmap, int c0, int c1, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
      ::"r"(smem_dst), "l"(tmap), "r"(c0), "r"(c1), "r"(bar)
      : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(uint64_t tmap) {
  asm volatile("prefetch.tensormap [%0];" ::"l"(tmap) : "memory");
}

__device__ __forceinline__ void tcgen05_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tcgen05_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

__device__ __forceinline__ void tmem_alloc(uint32_t smem_dst, uint32_t cols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(cols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t cols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
}

// D[tmem] (+)= A[smem] * B[smem]; issued by ONE thread on behalf of the CTA.
__device__ __forceinline__ void umma_f16(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
// mbarrier arrives once every tcgen05.mma issued so far by this thread has completed (implies fence::before_thread_sync).
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}

// 32 lanes x 32 consecutive fp32 columns: thread t of the warp receives row (lane base + t), columns [col, col + 32).
__device__ __forceinline__ void tmem_ld_32x32(uint32_t taddr, uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
        "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]),
        "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]),
        "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
      : "r"(taddr)
      : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// ------------------------------------------------------------------------------------------------ descriptors
// Shared-memory matrix descriptor (PTX ISA "tcgen05 shared memory descriptor"): start address >> 4 in bits [0,14),
// leading byte offset >> 4 in [16,30), stride byte offset >> 4 in [32,46), version 1 in [46,48), swizzle mode in
// [61,64) (2 = 128-byte swizzle).  Tiles are 128-byte rows grouped in 8-row (1024 B) swizzle atoms.
constexpr uint32_t kDescHi = (1024u >> 4) | (1u << 14) | (2u << 29);   // SBO = 1024 B, version 1, SWIZZLE_128B

// K-major operand: row r of the tile at byte r * 128; the K offset inside the 128-byte row is added to the address.
__device__ __forceinline__ uint64_t desc_kmajor(uint32_t saddr) {
  const uint32_t lo = ((saddr >> 4) & 0x3FFFu) | (1u << 16);            // LBO unused for swizzled K-major (set to 1)
  return (static_cast<uint64_t>(kDescHi) << 32) | lo;
}
// MN-major operand (B of OP_BX): 64 K rows x 128 B per 64-wide N chunk; next N chunk LBO = 8192 B further,
// next group of 8 K rows SBO = 1024 B further.
__device__ __forceinline__ uint64_t desc_mnmajor(uint32_t saddr) {
  const uint32_t lo = ((saddr >> 4) & 0x3FFFu) | ((8192u >> 4) << 16);
  return (static_cast<uint64_t>(kDescHi) << 32) | lo;
}
// Instruction descriptor for kind::f16: D = fp32 (bits [4,6) = 1), A/B format fp16 (0) in [7,10)/[10,13),
// B major-ness in bit 16 (1 = MN-major), N >> 3 in [17,23), M >> 4 in [24,29).
__device__ __forceinline__ uint32_t make_idesc(int n, bool b_mn_major) {
  return (1u << 4) | (static_cast<uint32_t>(b_mn_major) << 16) | (static_cast<uint32_t>(n >> 3) << 17) |
         (static_cast<uint32_t>(kBlk >> 4) << 24);
}

__device__ __forceinline__ uint32_t pack_half2(float lo, float hi) {
  __half2 h = __floats2half2_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&h);
}

// ------------------------------------------------------------------------------------------------ the kernel
template <int kOp>
__global__ void __launch_bounds__(kNumThreads, 1)
ns_gemm_kernel(const GemmProblem* __restrict__ probs, const TileUnit* __restrict__ units, int units_per_problem,
               int total_units, int k_blocks, float alpha, float beta) {
  constexpr bool kSym = (kOp != OP_BX);
  constexpr bool kBMn = (kOp == OP_BX);
  constexpr bool kAddend = (kOp != OP_SYRK);

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

  if (threadIdx.x == 0) {
    for (int s = 0; s < kStages; ++s) {
      mbar_init(bar_full + 8 * s, 1);
      mbar_init(bar_empty + 8 * s, 1);
    }
    for (int s = 0; s < 2; ++s) {
      mbar_init(bar_tfull + 8 * s, 1);
      mbar_init(bar_tempty + 8 * s, 128);
    }
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc(ctl_addr + offsetof(SmemCtl, tmem_base), kTmemCols);
  tcgen05_fence_before();
  __syncthreads();
  tcgen05_fence_after();
  const uint32_t tmem_base = ctl->tmem_base;

  if (warp == 0) {
    // ================================================================== TMA producer
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      for (int u = blockIdx.x; u < total_units; u += gridDim.x) {
        const int p = u / units_per_problem;
        const TileUnit tu = units[u - p * units_per_problem];
        const GemmProblem* pr = probs + p;
        const uint64_t tmA = reinterpret_cast<uint64_t>(&pr->tmA);
        const uint64_t tmB = reinterpret_cast<uint64_t>(&pr->tmB);
        const int w = tu.width;
        const uint32_t tx = kABytes + w * kBBlockBytes;
        for (int kb = 0; kb < k_blocks; ++kb) {
          mbar_wait(bar_empty + 8 * stage, phase ^ 1);
          const uint32_t fb = bar_full + 8 * stage;
          mbar_expect_tx(fb, tx);
          const uint32_t sA = base + stage * kStageBytes;
          const uint32_t sB = sA + kABytes;
          tma_load_2d(sA, tmA, kb * kBlkK, tu.m_blk * kBlk, fb);
          if (!kBMn) {
            for (int q = 0; q < w; ++q) tma_load_2d(sB + q * kBBlockBytes, tmB, kb * kBlkK, (tu.n_blk + q) * kBlk, fb);
          } else {
            for (int q = 0; q < 2 * w; ++q)   // 64 (n) x 64 (k) boxes, 8 KB each
              tma_load_2d(sB + q * (kBBlockBytes / 2), tmB, tu.n_blk * kBlk + q * 64, kb * kBlkK, fb);
          }
          if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
      }
    }
    __syncwarp();
  } else if (warp == 1) {
    // ================================================================== MMA issuer
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      int it = 0;
      for (int u = blockIdx.x; u < total_units; u += gridDim.x, ++it) {
        const int p = u / units_per_problem;
        const TileUnit tu = units[u - p * units_per_problem];
        const uint32_t idesc = make_idesc(tu.width * kBlk, kBMn);
        const int as = it & 1;
        const uint32_t aphase = (it >> 1) & 1;
        mbar_wait(bar_tempty + 8 * as, aphase ^ 1);    // epilogue has drained this accumulator
        tcgen05_fence_after();
        const uint32_t d_tmem = tmem_base + as * kAccCols;
        for (int kb = 0; kb < k_blocks; ++kb) {
          mbar_wait(bar_full + 8 * stage, phase);       // TMA bytes have landed
          tcgen05_fence_after();
          const uint32_t sA = base + stage * kStageBytes;
          const uint32_t sB = sA + kABytes;
#pragma unroll
          for (int k = 0; k < kBlkK / 16; ++k) {
            const uint64_t ad = desc_kmajor(sA + k * 32);
            const uint64_t bd = kBMn ? desc_mnmajor(sB + k * 2048) : desc_kmajor(sB + k * 32);
            umma_f16(d_tmem, ad, bd, idesc, (kb | k) != 0);
          }
          umma_commit(bar_empty + 8 * stage);           // frees the smem slot when these MMAs finish
          if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
        umma_commit(bar_tfull + 8 * as);                // accumulator complete -> epilogue
      }
    }
    __syncwarp();
  } else {
    // ================================================================== epilogue (4 warps, one TMEM lane quarter each)
    const int q = warp & 3;
    const int row = q * 32 + lane;
    int it = 0;
    for (int u = blockIdx.x; u < total_units; u += gridDim.x, ++it) {
      const int p = u / units_per_problem;
      const TileUnit tu = units[u - p * units_per_problem];
      const GemmProblem* pr = probs + p;
      __half* __restrict__ C = pr->C;
      const __half* __restrict__ D = pr->D;
      const int64_t ldc = pr->ldc;
      const int as = it & 1;
      const uint32_t aphase = (it >> 1) & 1;
      mbar_wait(bar_tfull + 8 * as, aphase);
      tcgen05_fence_after();
      const uint32_t taddr = tmem_base + as * kAccCols + (static_cast<uint32_t>(q * 32) << 16);
      const int64_t grow = static_cast<int64_t>(tu.m_blk) * kBlk + row;
      const int chunks = tu.width * (kBlk / 32);
      for (int c = 0; c < chunks; ++c) {
        uint32_t v[32];
        tmem_ld_32x32(taddr + c * 32, v);
        tmem_wait_ld();
        if (c == chunks - 1) {                           // accumulator fully read: hand it back to the MMA warp
          tcgen05_fence_before();
          mbar_arrive(bar_tempty + 8 * as);
        }
        const int64_t gcol = static_cast<int64_t>(tu.n_blk) * kBlk + c * 32;
        uint32_t o[16];
        if (kAddend) {
          const uint4* dp = reinterpret_cast<const uint4*>(D + grow * ldc + gcol);
#pragma unroll
          for (int g = 0; g < 4; ++g) {
            const uint4 d4 = __ldg(dp + g);
            const uint32_t dw[4] = {d4.x, d4.y, d4.z, d4.w};
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              const float2 df = __half22float2(*reinterpret_cast<const __half2*>(&dw[e]));
              const float lo = fmaf(alpha, __uint_as_float(v[g * 8 + e * 2]), beta * df.x);
              const float hi = fmaf(alpha, __uint_as_float(v[g * 8 + e * 2 + 1]), beta * df.y);
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
        if (kSym && (tu.n_blk + (c >> 2)) != tu.m_blk) {
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
    }
  }

  tcgen05_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem_base, kTmemCols);
}

template <int kOp>
int launch_op(const GemmLaunch& L, cudaStream_t stream) {
  static bool configured = false;
  auto kern = ns_gemm_kernel<kOp>;
  if (!configured) {
    DMUON_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes));
    configured = true;
  }
  const int total = L.units_per_problem * L.num_problems;
  if (total <= 0) return DMUON_OK;
  const int grid = L.grid < total ? L.grid : total;
  kern<<<grid, kNumThreads, kSmemBytes, stream>>>(L.problems, L.units, L.units_per_problem, total, L.k_blocks,
                                                 L.alpha, L.beta);
  DMUON_CUDA_CHECK(cudaGetLastError());
  return DMUON_OK;
}

}  // namespace

int gemm_smem_bytes() { return kSmemBytes; }

int launch_ns_gemm(const GemmLaunch& L, cudaStream_t stream) {
  switch (L.op) {
    case OP_SYRK: return launch_op<OP_SYRK>(L, stream);
    case OP_SQ: return launch_op<OP_SQ>(L, stream);
    case OP_BX: return launch_op<OP_BX>(L, stream);
  }
  set_error("launch_ns_gemm: bad op %d", static_cast<int>(L.op));
  return DMUON_ERR_INVALID_ARG;
}

}  // namespace dmuon
