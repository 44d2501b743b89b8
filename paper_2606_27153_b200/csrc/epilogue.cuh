// What the LAST X update of a call does with its fp32 result x (one accumulator row, 32 consecutive columns per
// lane), shared by the grouped GEMM family (gemm_sm100.cu) and the on-chip small-matrix kernel (ns_small_sm100.cu):
//
//   EPI_BF16          out = bf16(x / c)                               the NS output of dmuon_ns_batched
//   EPI_APPLY         W' = bf16(W - (lr scale x / c + lr wd W))       step a6 (Eq. 1; readings N4, N5)
//   EPI_APPLY_MASTER  W32' = W32 - (...), W' = bf16(W32')             fp32 master weights
//
// ("elementwise operations ... fused into the same epilogue".)  Device code only.
#pragma once

#include <cstdint>
#include <cuda_bf16.h>

#include "common.h"

namespace dmuon {

// Destination of a fused final epilogue: the caller's tensors of the unit's matrix.
struct FinalCtx {
  uint16_t* W;        // bf16 parameter / output
  float* W32;         // fp32 master (EPI_APPLY_MASTER)
  int64_t ldw;        // leading dimension of W / W32, in elements
  float so;           // EPI_APPLY*: lr * scale / c ; EPI_BF16: 1 / c
};

__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  const __nv_bfloat162 b = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<const uint32_t*>(&b);
}

// W words of one 32-column chunk of one row (EPI_APPLY), loaded one chunk ahead.  Through L1 (ld.global.ca): a lane
// reads its row's 64 bytes as four 16-byte loads, the first brings the sectors in and the other three hit; a streaming
// load (ld.global.cs) sent all four to L2/DRAM and halved the throughput of the fused X update.  Not the read-only
// path (ld.global.nc / __ldg): the same kernel overwrites W in final_store, and .nc is defined only for memory that
// nobody writes while the kernel runs.
struct WWords { uint4 w[4]; };
template <int kEpi>
__device__ __forceinline__ void load_w(WWords& a, const FinalCtx& x, int64_t grow, int64_t gcol) {
  if (kEpi == EPI_APPLY) {
    const uint4* wp = reinterpret_cast<const uint4*>(x.W + grow * x.ldw + gcol);
#pragma unroll
    for (int g = 0; g < 4; ++g)
      asm volatile("ld.global.ca.v4.u32 {%0, %1, %2, %3}, [%4];"
                   : "=r"(a.w[g].x), "=r"(a.w[g].y), "=r"(a.w[g].z), "=r"(a.w[g].w)
                   : "l"(wp + g));
  }
}

// r = the 32 fp32 values x of row `grow`, columns [gcol, gcol + 32).
template <int kEpi>
__device__ __forceinline__ void final_store(const float (&r)[32], const WWords& ww, const FinalCtx& x, int64_t grow,
                                            int64_t gcol, float lrwd) {
  if (kEpi == EPI_BF16) {
    // NS output of dmuon_ns_batched: out = bf16(x / c), c a power of two
    uint32_t o[16];
#pragma unroll
    for (int e = 0; e < 16; ++e) o[e] = pack_bf16x2(r[2 * e] * x.so, r[2 * e + 1] * x.so);
    uint4* wp = reinterpret_cast<uint4*>(x.W + grow * x.ldw + gcol);
#pragma unroll
    for (int g = 0; g < 4; ++g) wp[g] = make_uint4(o[g * 4], o[g * 4 + 1], o[g * 4 + 2], o[g * 4 + 3]);
  } else if (kEpi == EPI_APPLY) {
    // a6: W' = W - (lr scale O + lr wd W), one fp32 expression, one RNE rounding
    uint32_t o[16];
#pragma unroll
    for (int g = 0; g < 4; ++g) {
      const uint32_t wd[4] = {ww.w[g].x, ww.w[g].y, ww.w[g].z, ww.w[g].w};
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const float w0 = __uint_as_float(wd[e] << 16), w1 = __uint_as_float(wd[e] & 0xFFFF0000u);
        const float t0 = fmaf(x.so, r[g * 8 + e * 2], lrwd * w0);
        const float t1 = fmaf(x.so, r[g * 8 + e * 2 + 1], lrwd * w1);
        o[g * 4 + e] = pack_bf16x2(w0 - t0, w1 - t1);
      }
    }
    uint4* wp = reinterpret_cast<uint4*>(x.W + grow * x.ldw + gcol);
#pragma unroll
    for (int g = 0; g < 4; ++g) wp[g] = make_uint4(o[g * 4], o[g * 4 + 1], o[g * 4 + 2], o[g * 4 + 3]);
  } else if (kEpi == EPI_APPLY_MASTER) {
    // fp32 master weights: the update lands in the master, the bf16 parameter is its rounding
    float4* mp = reinterpret_cast<float4*>(x.W32 + grow * x.ldw + gcol);
    uint32_t o[16];
#pragma unroll
    for (int g = 0; g < 8; ++g) {
      const float4 w = mp[g];
      float4 n;
      n.x = w.x - fmaf(x.so, r[g * 4], lrwd * w.x);
      n.y = w.y - fmaf(x.so, r[g * 4 + 1], lrwd * w.y);
      n.z = w.z - fmaf(x.so, r[g * 4 + 2], lrwd * w.z);
      n.w = w.w - fmaf(x.so, r[g * 4 + 3], lrwd * w.w);
      mp[g] = n;
      o[g * 2] = pack_bf16x2(n.x, n.y);
      o[g * 2 + 1] = pack_bf16x2(n.z, n.w);
    }
    uint4* wp = reinterpret_cast<uint4*>(x.W + grow * x.ldw + gcol);
#pragma unroll
    for (int g = 0; g < 4; ++g) wp[g] = make_uint4(o[g * 4], o[g * 4 + 1], o[g * 4 + 2], o[g * 4 + 3]);
  }
}

}  // namespace dmuon
