// On-chip Newton-Schulz for small matrices on sm_100a: ALL k steps of one 256 x 256 (padded) matrix in one kernel,
// X, G and B resident in the shared memory of a CTA pair from the first load to the last epilogue (Eq. 2 in
// the Gram form of PAPER.md:170; "batched by shape"; PAPER.md:182 fused epilogues).
//
// Why: with the per-product grouped launches of gemm_sm100.cu a bucket of many small matrices streams every
// intermediate (G, B, X') through HBM -- 15 products x ~0.3 MB per 256 x 256 matrix, 315 GB for the 65 536 matrices
// of configs[4] -- and each 256 x 256 unit's epilogue (TMEM -> registers -> shared -> TMA store, plus the mirrored
// tile and the addend loads) costs more than its 16 MMAs.  Here a matrix is read once (128 KB fp16) and written once.
//
// One CTA pair (cluster of 2, one TPC) per matrix, cta_group::2 UMMA M = 256, N = 256, K = 16.  CTA r owns rows
// [128 r, 128 r + 128) of X, G, B and of every accumulator (its own TMEM, 2 x 256 columns).  Shared memory of CTA r:
//
//   XR  X[own rows, all cols]   4 K-major tiles (128 rows x 64 cols, 128-byte swizzle)   A and B operand of G = X X^T,
//                                                                                        addend of X' = a X + B X
//   XC  X[all rows, own cols]   2 MN-major panels (256 rows x 64 cols)                   B operand of B X (N = own cols)
//   AB  G, then B in place      4 K-major tiles                                          both operands of G G, A operand of B X
//
// Both CTAs hold contraction block kb at the same offset (cta_group::2 descriptors are per-pair).  The epilogue warps
// write the next product's operands straight into these tiles (st.shared); the copy engine (cp.async.bulk shared ->
// shared::cluster) then moves each finished 16 KB tile of X' into the MN-major panel of the CTA that owns those
// columns, so no product touches global memory and no thread waits for a remote store.  The chain of 3 k products is serial per
// matrix, but it is pipelined at tile granularity: the epilogue signals "tile kb written" after every 64 columns and
// the MMA thread starts contraction block kb of the NEXT product as soon as both CTAs have written it, into the other
// TMEM accumulator.  Symmetry of G and B is not exploited (the tensor pipe is not the bound here; the epilogue is).
//
// The last X update writes from registers: fp16 X_k (EPI_F16 / store_c) and/or the fused final epilogues of
// epilogue.cuh (bf16 NS output, Muon update on bf16 weights or fp32 masters).
#include <cstring>

#include "common.h"
#include "epilogue.cuh"
#include "umma.cuh"

namespace dmuon {
namespace {

using namespace umma;

constexpr int kTileBytes = 128 * 128;       // 16 KB: 128 rows x 64 fp16
constexpr int kPanelBytes = 256 * 128;      // 32 KB: 256 rows x 64 fp16
constexpr int kXR = 0;                      // 4 tiles
constexpr int kXC = 4 * kTileBytes;         // 2 panels
constexpr int kAB = kXC + 2 * kPanelBytes;  // 4 tiles
constexpr int kOperandBytes = kAB + 4 * kTileBytes;   // 192 KB
// Epilogue warps: kSub per TMEM lane quarter.  The chain of products of one matrix is serial, so the time between two
// products is the epilogue's LATENCY, not its throughput: sub-warp j of a quarter takes the 32-column chunks j, j + kSub,
// ... of its 32 rows, so that 16 warps finish a 128 x 256 accumulator in two chunk times.
#ifndef DMUON_SMALL_SUB
#define DMUON_SMALL_SUB 4
#endif
constexpr int kSub = DMUON_SMALL_SUB;
constexpr int kSmallEpiWarps = 4 * kSub;
constexpr int kSmallThreads = 64 + 32 * kSmallEpiWarps;   // warp 0: TMA, warp 1: MMA (leader) + TMEM owner, then the epilogue warps
static_assert(kSub == 1 || kSub == 2 || kSub == 4, "sub-warps per quarter");

struct SmallCtl {
  uint64_t x_full;          // leader's: both CTAs' X tiles of the current matrix have landed
  uint64_t x_free;          // own: this CTA's epilogue warps have read their last addend from XR (current matrix)
  uint64_t xc_free;         // own: the last MMA of the current matrix has read XC (tcgen05.commit, multicast)
  uint64_t ready[4];        // leader's: contraction tile kb of the next product's operands is written (16 chunk arrivals:
                            // 2 chunks x 4 lane quarters x 2 CTAs)
  uint64_t tfull[2];        // own: accumulator stage complete (tcgen05.commit, multicast to both CTAs)
  uint64_t xc_full;         // own: the four 16 KB tiles of X' (two from each CTA) have landed in this CTA's XC panels
  uint64_t pxc_ready;       // leader's: the PEER's xc_full completed (relayed by the peer's otherwise idle warp 1)
  uint32_t tile_cnt[4];     // own: chunk writers of XR tile kb so far (8 per X update)
  uint32_t tmem_base;
  uint32_t pad;
};
constexpr int kSmallSmem = kOperandBytes + 256 + 1024;
static_assert(sizeof(SmallCtl) <= 256 && kSmallSmem <= 232448, "shared memory budget");

struct alignas(64) SmallParams {
  CUtensorMap tmX;          // 3-D: {256 cols, 256 rows, slots} of the bucket's X0 buffers, box {64, 128, 1}, 128-byte swizzle
  uint16_t* out;            // fp16 result of slot k at out + k * slot_elems, row stride 256
  uint64_t slot_elems;
  const MatRec* recs;
  int rec_base, count, steps, store_c;
  float gram_alpha, lr, lrwd, pad;
  float poly_alpha[kSmallMaxSteps], poly_beta[kSmallMaxSteps], x_beta[kSmallMaxSteps];
};

enum Kind : int { KIND_GRAM = 0, KIND_POLY = 1, KIND_X = 2, KIND_X_FINAL = 3 };

// One product's epilogue for this warp's 32 rows and its chunks c = sub, sub + kSub, ... of 32 columns; after every
// chunk the leader's MMA thread is told that a part of contraction tile kb = c / 2 of the next product's operand is written.
template <int kKind, int kEpi>
__device__ __forceinline__ void epi_product(uint32_t taddr, uint32_t smem, uint32_t cnt_addr, uint32_t xcfull_addr, int i, int sub,
                                            uint32_t rank, uint32_t ready_leader,
                                            float alpha, float beta, const FinalCtx& fin, uint16_t* out_row,
                                            int64_t grow, float lrwd, int store_c) {
  const int lane = threadIdx.x & 31;
  const uint32_t sw = static_cast<uint32_t>(i) & 7u;
  const uint32_t row_off = static_cast<uint32_t>(i) * 128u;
  WWords ww = {};
#pragma unroll 1
  for (int c = sub; c < 8; c += kSub) {
    uint32_t v[32];
    tmem_ld_32x32(taddr + c * 32, v);
    if (kKind == KIND_X_FINAL) load_w<kEpi>(ww, fin, grow, c * 32);
    const int kb = c >> 1;
    const uint32_t ch0 = (c & 1) * 4;
    // addend (in place): G for the polynomial, X for the X update
    uint4 d[4];
    if (kKind != KIND_GRAM) {
      const uint32_t src = smem + (kKind == KIND_POLY ? kAB : kXR) + kb * kTileBytes + row_off;
#pragma unroll
      for (int g = 0; g < 4; ++g) d[g] = ld_shared_v4(src + (((ch0 + g) ^ sw) << 4));
    }
    tmem_wait_ld();
    float r[32];
    if (kKind == KIND_GRAM) {
#pragma unroll
      for (int e = 0; e < 32; ++e) r[e] = alpha * __uint_as_float(v[e]);
    } else {
#pragma unroll
      for (int g = 0; g < 4; ++g) {
        const uint32_t dw[4] = {d[g].x, d[g].y, d[g].z, d[g].w};
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const float2 df = __half22float2(*reinterpret_cast<const __half2*>(&dw[e]));
          r[g * 8 + e * 2] = fmaf(alpha, __uint_as_float(v[g * 8 + e * 2]), beta * df.x);
          r[g * 8 + e * 2 + 1] = fmaf(alpha, __uint_as_float(v[g * 8 + e * 2 + 1]), beta * df.y);
        }
      }
    }
    if (kKind != KIND_X_FINAL) {
      uint32_t o[16];
#pragma unroll
      for (int e = 0; e < 16; ++e) o[e] = pack_half2(r[2 * e], r[2 * e + 1]);
      const uint32_t dst = smem + (kKind == KIND_X ? kXR : kAB) + kb * kTileBytes + row_off;
#pragma unroll
      for (int g = 0; g < 4; ++g) st_shared_v4(dst + (((ch0 + g) ^ sw) << 4), o[g * 4], o[g * 4 + 1], o[g * 4 + 2], o[g * 4 + 3]);
    } else {
      if (kEpi == EPI_F16 || store_c) {
        uint4* op = reinterpret_cast<uint4*>(out_row + c * 32);
#pragma unroll
        for (int g = 0; g < 4; ++g)
          op[g] = make_uint4(pack_half2(r[g * 8], r[g * 8 + 1]), pack_half2(r[g * 8 + 2], r[g * 8 + 3]),
                             pack_half2(r[g * 8 + 4], r[g * 8 + 5]), pack_half2(r[g * 8 + 6], r[g * 8 + 7]));
      }
      if (kEpi != EPI_F16) final_store<kEpi>(r, ww, fin, grow, c * 32, lrwd);
    }
    // this warp's part of tile kb is written (and these accumulator columns are read)
    fence_proxy_async();
    tcgen05_fence_before();
    __syncwarp();
    if (lane == 0) {
      mbar_arrive_cluster(ready_leader + 8 * kb);
      if (kKind == KIND_X) {
        // The CTA that owns columns [64 kb, +64) needs these 128 rows in its MN-major panel (operand of the NEXT X
        // update): the last of this CTA's 8 chunk writers of the tile hands the whole 16 KB tile to the copy engine
        // (st.shared::cluster from the epilogue registers cost 1.5 us per X update: profiles/r2_small_fused.md).
        const uint32_t old = atom_add_acqrel_shared(cnt_addr + 4 * kb, 1u);
        if ((old & 7u) == 7u) {
          const uint32_t owner = static_cast<uint32_t>(kb) >> 1;
          const uint32_t dst = mapa(smem + kXC + (kb & 1) * kPanelBytes + rank * kTileBytes, owner);
          bulk_copy_to_cluster(dst, smem + kXR + kb * kTileBytes, kTileBytes, mapa(xcfull_addr, owner));
        }
      }
    }
  }
}

template <int kEpi>
__global__ void __launch_bounds__(kSmallThreads, 1) ns_small_fused_kernel(const __grid_constant__ SmallParams p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t smem = (raw + 1023u) & ~1023u;
  const uint32_t ctl_addr = smem + kOperandBytes;
  SmallCtl* ctl = reinterpret_cast<SmallCtl*>(smem_raw + (ctl_addr - raw));
  const uint32_t bar_xfull = ctl_addr + offsetof(SmallCtl, x_full);
  const uint32_t bar_xfree = ctl_addr + offsetof(SmallCtl, x_free);
  const uint32_t bar_xcfree = ctl_addr + offsetof(SmallCtl, xc_free);
  const uint32_t bar_ready = ctl_addr + offsetof(SmallCtl, ready);
  const uint32_t bar_tfull = ctl_addr + offsetof(SmallCtl, tfull);
  const uint32_t bar_xcfull = ctl_addr + offsetof(SmallCtl, xc_full);
  const uint32_t bar_pxc = ctl_addr + offsetof(SmallCtl, pxc_ready);
  const uint32_t bar_cnt = ctl_addr + offsetof(SmallCtl, tile_cnt);

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const int worker = blockIdx.x >> 1;
  const int num_workers = gridDim.x >> 1;

  if (threadIdx.x == 0) {
    mbar_init(bar_xfull, 1);
    mbar_init(bar_xfree, kSmallEpiWarps);
    mbar_init(bar_xcfree, 1);
    mbar_init(bar_xcfull, 1);
    mbar_init(bar_pxc, 1);
    for (int k = 0; k < 4; ++k) ctl->tile_cnt[k] = 0;
    for (int k = 0; k < 4; ++k) mbar_init(bar_ready + 8 * k, 16);
    for (int s = 0; s < 2; ++s) mbar_init(bar_tfull + 8 * s, 1);
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc<2>(ctl_addr + offsetof(SmallCtl, tmem_base), 512);
  tcgen05_fence_before();
  cluster_sync();
  tcgen05_fence_after();
  const uint32_t tmem_base = ctl->tmem_base;

  if (warp == 0) {
    // ================================================================== TMA: this CTA's X tiles of each of its matrices
    if (lane == 0) {
      const uint64_t tm = reinterpret_cast<uint64_t>(&p.tmX);
      const uint32_t fb = mapa(bar_xfull, 0);
      int mi = 0;
      for (int k = worker; k < p.count; k += num_workers, ++mi) {
        const int r0 = 128 * static_cast<int>(rank);
        // XC was last read by the previous matrix's last MMA: the panels are refilled while the last epilogue runs.  (One
        // barrier phase per matrix: a parity wait on tfull would be fooled, this thread runs many phases ahead of it.)
        if (mi > 0) mbar_wait(bar_xcfree, (mi - 1) & 1);
        // (after the wait: the previous matrix's phase of x_full completed long before its last product)
        if (rank == 0) mbar_expect_tx(bar_xfull, 2 * (4 * kTileBytes + 2 * kPanelBytes));
        for (int q = 0; q < 2; ++q) {
          tma_load_3d_pair(smem + kXC + q * kPanelBytes, tm, r0 + 64 * q, 0, k, fb);
          tma_load_3d_pair(smem + kXC + q * kPanelBytes + kTileBytes, tm, r0 + 64 * q, 128, k, fb);
        }
        if (mi > 0) mbar_wait(bar_xfree, (mi - 1) & 1);       // the last epilogue has read its addend from XR
        for (int kb = 0; kb < 4; ++kb) tma_load_3d_pair(smem + kXR + kb * kTileBytes, tm, 64 * kb, r0, k, fb);
      }
    }
    __syncwarp();
  } else if (warp == 1) {
    // ================================================================== MMA issuer (leader CTA)
    if (lane == 0 && rank == 0) {
      const uint32_t idesc_kk = make_idesc(256, 256, false, false);
      const uint32_t idesc_kn = make_idesc(256, 256, false, true);
      uint32_t P = 0, Q = 0;     // products so far; X updates whose result went to the XC panels so far
      int mi = 0;
      for (int k = worker; k < p.count; k += num_workers, ++mi) {
        mbar_wait(bar_xfull, mi & 1);
        for (int s = 0; s < p.steps; ++s) {
          for (int t = 0; t < 3; ++t, ++P) {
            const uint32_t d_tmem = tmem_base + (P & 1) * 256;
            const uint32_t a_base = smem + (t == 0 ? kXR : kAB);
            if (t == 2 && s > 0) {
              // the previous X update's tiles have landed in both CTAs' XC panels (copy engine; two products ago)
              mbar_wait(bar_xcfull, Q & 1);
              mbar_wait_cluster(bar_pxc, Q & 1);
              ++Q;
            }
            for (int kb = 0; kb < 4; ++kb) {
              // both CTAs' epilogue warps have written contraction tile kb (and, at kb = 3, drained the accumulator
              // this product's successor will overwrite)
              if (P > 0) mbar_spin_wait<true>(bar_ready + 8 * kb, (P - 1) & 1);
              tcgen05_fence_after();
#pragma unroll
              for (int j = 0; j < 4; ++j) {
                const uint64_t ad = desc_kmajor(a_base + kb * kTileBytes + j * 32);
                const uint64_t bd = t == 2 ? desc_mnmajor_lbo(smem + kXC + kb * 8192 + j * 2048, kPanelBytes)
                                           : desc_kmajor(a_base + kb * kTileBytes + j * 32);
                mma_f16<2>(d_tmem, ad, bd, t == 2 ? idesc_kn : idesc_kk, (kb | j) != 0);
              }
            }
            mma_commit_pair(bar_tfull + 8 * (P & 1), 3);
          }
        }
        mma_commit_pair(bar_xcfree, 3);
      }
    } else if (lane == 0) {
      // peer CTA: tell the leader's MMA thread when this CTA's XC panels hold the new X
      const uint32_t pxc_leader = mapa(bar_pxc, 0);
      uint32_t Q = 0;
      for (int k = worker; k < p.count; k += num_workers)
        for (int s = 0; s + 1 < p.steps; ++s, ++Q) {
          mbar_wait(bar_xcfull, Q & 1);
          mbar_arrive_cluster(pxc_leader);
        }
    }
    __syncwarp();
  } else {
    // ================================================================== epilogue (TMEM lane quarter warp % 4)
    const int q = warp & 3;
    const int sub = (warp - 2) >> 2;                  // which of the quarter's chunks this warp takes
    const int i = q * 32 + lane;                      // row inside this CTA's 128
    const uint32_t ready_leader = mapa(bar_ready, 0);
    uint32_t P = 0;
    for (int k = worker; k < p.count; k += num_workers) {
      const int64_t grow = 128 * static_cast<int64_t>(rank) + i;
      FinalCtx fin;
      fin.W = nullptr; fin.W32 = nullptr; fin.ldw = 256; fin.so = 0.f;
      if (kEpi != EPI_F16) {
        const MatRec& rec = p.recs[p.rec_base + k];
        fin.W = static_cast<uint16_t*>(rec.W);
        fin.W32 = rec.W32;
        fin.so = kEpi == EPI_BF16 ? rec.inv_xscale : p.lr * rec.scale * rec.inv_xscale;
      }
      uint16_t* out_row = p.out + static_cast<uint64_t>(k) * p.slot_elems + grow * 256;
      for (int s = 0; s < p.steps; ++s) {
        for (int t = 0; t < 3; ++t, ++P) {
          mbar_spin_wait<false>(bar_tfull + 8 * (P & 1), (P >> 1) & 1);
          tcgen05_fence_after();
          const uint32_t taddr = tmem_base + (P & 1) * 256 + (static_cast<uint32_t>(q * 32) << 16);
          if (t == 0) epi_product<KIND_GRAM, kEpi>(taddr, smem, bar_cnt, bar_xcfull, i, sub, rank, ready_leader, p.gram_alpha, 0.f, fin, out_row, grow, p.lrwd, p.store_c);
          else if (t == 1) epi_product<KIND_POLY, kEpi>(taddr, smem, bar_cnt, bar_xcfull, i, sub, rank, ready_leader, p.poly_alpha[s], p.poly_beta[s], fin, out_row, grow, p.lrwd, p.store_c);
          else if (s + 1 < p.steps) {
            // this CTA's XC panels will receive the new X: two tiles from each CTA's copy engine
            if (warp == 2 && lane == 0) mbar_expect_tx(bar_xcfull, 4 * kTileBytes);
            epi_product<KIND_X, kEpi>(taddr, smem, bar_cnt, bar_xcfull, i, sub, rank, ready_leader, 1.f, p.x_beta[s], fin, out_row, grow, p.lrwd, p.store_c);
          } else {
            epi_product<KIND_X_FINAL, kEpi>(taddr, smem, bar_cnt, bar_xcfull, i, sub, rank, ready_leader, 1.f, p.x_beta[s], fin, out_row, grow, p.lrwd, p.store_c);
          }
        }
      }
      // XR (the last addend) and XC are free for the next matrix
      __syncwarp();
      if (lane == 0) mbar_arrive(bar_xfree);
    }
  }

  tcgen05_fence_before();
  cluster_sync();
  if (warp == 1) tmem_dealloc<2>(tmem_base, 512);
}

typedef void (*SmallKernel)(const SmallParams);
SmallKernel g_small[kNumEpi] = {ns_small_fused_kernel<EPI_F16>, ns_small_fused_kernel<EPI_BF16>,
                                ns_small_fused_kernel<EPI_APPLY>, ns_small_fused_kernel<EPI_APPLY_MASTER>};
bool g_small_configured[kNumEpi][kMaxDevices];

}  // namespace

int launch_ns_small(const SmallLaunch& L, cudaStream_t stream) {
  if (L.steps < 1 || L.steps > kSmallMaxSteps || L.epi < 0 || L.epi >= kNumEpi) {
    set_error("launch_ns_small: bad step count %d / epilogue %d", L.steps, static_cast<int>(L.epi));
    return DMUON_ERR_INVALID_ARG;
  }
  if (L.count <= 0) return DMUON_OK;
  if (L.epi != EPI_F16 && !L.recs) { set_error("launch_ns_small: fused epilogue without matrix records"); return DMUON_ERR_INVALID_ARG; }
  int dev = 0;
  DMUON_CUDA_CHECK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) { set_error("launch_ns_small: device ordinal %d is not supported", dev); return DMUON_ERR_UNSUPPORTED_DEVICE; }
  SmallKernel kern = g_small[L.epi];
  if (!g_small_configured[L.epi][dev]) {
    DMUON_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmallSmem));
    g_small_configured[L.epi][dev] = true;
  }
  SmallParams p;
  memset(&p, 0, sizeof p);
  p.tmX = *L.tmX;
  p.out = static_cast<uint16_t*>(L.out);
  p.slot_elems = L.slot_bytes / 2;
  p.recs = L.recs;
  p.rec_base = L.rec_base;
  p.count = L.count;
  p.steps = L.steps;
  p.store_c = L.store_c ? 1 : 0;
  p.gram_alpha = L.gram_alpha;
  p.lr = L.lr;
  p.lrwd = L.lrwd;
  for (int s = 0; s < L.steps; ++s) {
    p.poly_alpha[s] = L.poly_alpha[s];
    p.poly_beta[s] = L.poly_beta[s];
    p.x_beta[s] = L.x_beta[s];
  }
  const int workers = L.grid / 2 < L.count ? L.grid / 2 : L.count;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(2 * workers);
  cfg.blockDim = dim3(kSmallThreads);
  cfg.dynamicSmemBytes = kSmallSmem;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = 2;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  DMUON_CUDA_CHECK(cudaLaunchKernelEx(&cfg, kern, p));
  return DMUON_OK;
}

}  // namespace dmuon
