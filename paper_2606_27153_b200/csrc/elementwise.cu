// HBM-bound kernels of the Muon step (DESIGN.md steps a1, a2, a6 and the orientation/normalisation pass):
//
//   momentum_kernel   M' = mu M + G ; U = bf16(G + mu M') ; per-chunk sum of squares of the rounded U   (a1 + a2)
//   sumsq_kernel      per-chunk sum of squares of a bf16 matrix                                          (a2 alone)
//   finalize_norms    1 / (||U||_F + eps) per matrix, fixed-order (deterministic) second reduction stage
//   normalize_kernel  X0 = U / (||U||_F + eps), transposed when rows > cols, zero padded to the
//                     128-multiples the GEMM tiles want, cast to the internal dtype (fp16, or fp32 in check mode)
//   apply_kernel      W' = W - lr (scale O + wd W)  (a6; Eq. 1)  /  out = bf16(O) for dmuon_ns_batched
//
// All global accesses are 128-bit and coalesced on the fast path (cols % 8 == 0); other shapes take a scalar path.
// Work is cut into fixed-size chunks/tiles over ALL matrices of the call, so one launch covers the whole set.
#include "common.h"

namespace dmuon {
namespace {

constexpr int kThreads = 256;

__device__ __forceinline__ int find_matrix(const int64_t* __restrict__ prefix, int count, int64_t id) {
  int lo = 0, hi = count;           // invariant: prefix[lo] <= id < prefix[hi]
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (__ldg(prefix + mid) <= id) lo = mid; else hi = mid;
  }
  return lo;
}

__device__ __forceinline__ float bf16_bits_to_float(uint32_t b) { return __uint_as_float(b << 16); }
__device__ __forceinline__ uint32_t float_to_bf16_bits(float f) {
  return static_cast<uint32_t>(__bfloat16_as_ushort(__float2bfloat16_rn(f)));
}
__device__ __forceinline__ float2 bf16x2_to_float2(uint32_t w) {
  return make_float2(__uint_as_float(w << 16), __uint_as_float(w & 0xFFFF0000u));
}
__device__ __forceinline__ uint32_t float2_to_bf16x2(float2 f) {
  const __nv_bfloat162 b = __floats2bfloat162_rn(f.x, f.y);     // .x in the low half
  return *reinterpret_cast<const uint32_t*>(&b);
}
__device__ __forceinline__ void unpack8(const uint4& v, float (&f)[8]) {
  const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    f[2 * i] = __uint_as_float(w[i] << 16);
    f[2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u);
  }
}
__device__ __forceinline__ uint4 pack8_bf16(const float (&f)[8]) {
  uint32_t w[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) w[i] = float_to_bf16_bits(f[2 * i]) | (float_to_bf16_bits(f[2 * i + 1]) << 16);
  return make_uint4(w[0], w[1], w[2], w[3]);
}

__device__ __forceinline__ float block_sum(float v, float* red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  __syncthreads();
  if (lane == 0) red[warp] = v;
  __syncthreads();
  float t = 0.f;
  if (threadIdx.x == 0) {
#pragma unroll
    for (int w = 0; w < kThreads / 32; ++w) t += red[w];   // fixed order
  }
  return t;
}

// ---------------------------------------------------------------------------------------------- a1 + a2
// kMomentum: read G, M; write M' (in place) and U; accumulate |bf16(U)|^2.   !kMomentum: accumulate |X|^2 of rec.W.
template <bool kMomentum>
__global__ void __launch_bounds__(kThreads) flat_kernel(const MatRec* __restrict__ recs,
                                                        const int64_t* __restrict__ prefix, int count,
                                                        int64_t total_chunks, float mu, float* __restrict__ partials) {
  __shared__ float red[kThreads / 32];
  constexpr int kIter = kFlatChunk / (kThreads * 8);   // 4
  for (int64_t chunk = blockIdx.x; chunk < total_chunks; chunk += gridDim.x) {
    const int mat = find_matrix(prefix, count, chunk);
    const MatRec& rec = recs[mat];
    const int64_t elems = static_cast<int64_t>(rec.rows) * rec.cols;
    const int64_t start = (chunk - __ldg(prefix + mat)) * kFlatChunk;
    const int64_t end = min(start + static_cast<int64_t>(kFlatChunk), elems);
    float acc = 0.f;
    float2 acc2 = make_float2(0.f, 0.f);
    const float2 mu2 = make_float2(mu, mu);
    if (kMomentum) {
      const uint16_t* __restrict__ G = static_cast<const uint16_t*>(rec.G);
      uint16_t* __restrict__ M = static_cast<uint16_t*>(rec.M);
      uint16_t* __restrict__ U = static_cast<uint16_t*>(rec.U);
      uint4 g4[kIter], m4[kIter];
#pragma unroll
      for (int it = 0; it < kIter; ++it) {          // all loads first: 8 x 16 B in flight per thread
        const int64_t i = start + (static_cast<int64_t>(it) * kThreads + threadIdx.x) * 8;
        if (i + 8 <= end) {
          g4[it] = __ldcs(reinterpret_cast<const uint4*>(G + i));
          m4[it] = __ldcs(reinterpret_cast<const uint4*>(M + i));
        }
      }
#pragma unroll
      for (int it = 0; it < kIter; ++it) {
        const int64_t i = start + (static_cast<int64_t>(it) * kThreads + threadIdx.x) * 8;
        if (i + 8 <= end) {
          // two elements per instruction: fma.rn.f32x2 and cvt.rn.bf16x2.f32 (same roundings as the scalar forms)
          const uint32_t gw[4] = {g4[it].x, g4[it].y, g4[it].z, g4[it].w};
          const uint32_t mw[4] = {m4[it].x, m4[it].y, m4[it].z, m4[it].w};
          uint32_t mo[4], uo[4];
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const float2 gf = bf16x2_to_float2(gw[e]);
            const float2 mf = bf16x2_to_float2(mw[e]);
            const float2 mn = __ffma2_rn(mu2, mf, gf);            // M' = mu M + G
            const float2 uf = __ffma2_rn(mu2, mn, gf);            // U  = G + mu M'   (from the unrounded M')
            mo[e] = float2_to_bf16x2(mn);
            uo[e] = float2_to_bf16x2(uf);
            const float2 ur = bf16x2_to_float2(uo[e]);            // the rounded U is what the norm is taken of
            acc2 = __ffma2_rn(ur, ur, acc2);
          }
          *reinterpret_cast<uint4*>(M + i) = make_uint4(mo[0], mo[1], mo[2], mo[3]);
          *reinterpret_cast<uint4*>(U + i) = make_uint4(uo[0], uo[1], uo[2], uo[3]);
        } else {
          for (int64_t j = i; j < end; ++j) {       // ragged tail of the matrix
            const float g = bf16_bits_to_float(G[j]), m = bf16_bits_to_float(M[j]);
            const float mn = fmaf(mu, m, g);
            const uint32_t ub = float_to_bf16_bits(fmaf(mu, mn, g));
            M[j] = static_cast<uint16_t>(float_to_bf16_bits(mn));
            U[j] = static_cast<uint16_t>(ub);
            const float uf = bf16_bits_to_float(ub);
            acc = fmaf(uf, uf, acc);
          }
        }
      }
    } else {
      const uint16_t* __restrict__ X = static_cast<const uint16_t*>(rec.W);
      uint4 x4[kIter];
#pragma unroll
      for (int it = 0; it < kIter; ++it) {
        const int64_t i = start + (static_cast<int64_t>(it) * kThreads + threadIdx.x) * 8;
        if (i + 8 <= end) x4[it] = __ldg(reinterpret_cast<const uint4*>(X + i));
      }
#pragma unroll
      for (int it = 0; it < kIter; ++it) {
        const int64_t i = start + (static_cast<int64_t>(it) * kThreads + threadIdx.x) * 8;
        if (i + 8 <= end) {
          const uint32_t xw[4] = {x4[it].x, x4[it].y, x4[it].z, x4[it].w};
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const float2 xf = bf16x2_to_float2(xw[e]);
            acc2 = __ffma2_rn(xf, xf, acc2);
          }
        } else {
          for (int64_t j = i; j < end; ++j) {
            const float x = bf16_bits_to_float(X[j]);
            acc = fmaf(x, x, acc);
          }
        }
      }
    }
    const float total = block_sum(acc + (acc2.x + acc2.y), red);
    if (threadIdx.x == 0) partials[chunk] = total;
  }
}

// One block per matrix: fixed-order sum of that matrix's chunk partials, in double.
__global__ void __launch_bounds__(kThreads) finalize_norms_kernel(const int64_t* __restrict__ prefix,
                                                                  const float* __restrict__ partials, float eps,
                                                                  float* __restrict__ inv_norm) {
  __shared__ double red[kThreads];
  const int mat = blockIdx.x;
  const int64_t b = prefix[mat], e = prefix[mat + 1];
  if (b == e) return;                     // matrix not in this launch's part (every member has at least one chunk)
  double acc = 0.0;
  for (int64_t i = b + threadIdx.x; i < e; i += kThreads) acc += static_cast<double>(partials[i]);
  red[threadIdx.x] = acc;
  __syncthreads();
  for (int s = kThreads / 2; s > 0; s >>= 1) {
    if (threadIdx.x < s) red[threadIdx.x] += red[threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x == 0) inv_norm[mat] = static_cast<float>(1.0 / (sqrt(red[0]) + static_cast<double>(eps)));
}

// ---------------------------------------------------------------------------------------------- 2-D tile helpers
template <typename T> struct Store8;
template <> struct Store8<__half> {
  static __device__ __forceinline__ void run(__half* p, const float (&f)[8]) {
    uint32_t w[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      __half2 h = __floats2half2_rn(f[2 * i], f[2 * i + 1]);
      w[i] = *reinterpret_cast<uint32_t*>(&h);
    }
    *reinterpret_cast<uint4*>(p) = make_uint4(w[0], w[1], w[2], w[3]);
  }
};
template <> struct Store8<float> {
  static __device__ __forceinline__ void run(float* p, const float (&f)[8]) {
    reinterpret_cast<float4*>(p)[0] = make_float4(f[0], f[1], f[2], f[3]);
    reinterpret_cast<float4*>(p)[1] = make_float4(f[4], f[5], f[6], f[7]);
  }
};
template <typename T> struct Load8;
template <> struct Load8<__half> {
  static __device__ __forceinline__ void run(const __half* p, float (&f)[8]) {
    const uint4 v = __ldg(reinterpret_cast<const uint4*>(p));
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const float2 t = __half22float2(*reinterpret_cast<const __half2*>(&w[i]));
      f[2 * i] = t.x;
      f[2 * i + 1] = t.y;
    }
  }
};
template <> struct Load8<float> {
  static __device__ __forceinline__ void run(const float* p, float (&f)[8]) {
    const float4 a = __ldg(reinterpret_cast<const float4*>(p));
    const float4 b = __ldg(reinterpret_cast<const float4*>(p) + 1);
    f[0] = a.x; f[1] = a.y; f[2] = a.z; f[3] = a.w;
    f[4] = b.x; f[5] = b.y; f[6] = b.z; f[7] = b.w;
  }
};

// Read 8 consecutive bf16 of row `r` starting at column `c` of a rows x cols matrix; zeros outside.
__device__ __forceinline__ void load8_bf16_guarded(const uint16_t* __restrict__ src, int rows, int cols, int r, int c,
                                                   bool vec_ok, float (&f)[8]) {
  if (r < rows && c + 8 <= cols && vec_ok) {
    unpack8(__ldg(reinterpret_cast<const uint4*>(src + static_cast<int64_t>(r) * cols + c)), f);
  } else {
#pragma unroll
    for (int e = 0; e < 8; ++e)
      f[e] = (r < rows && c + e < cols) ? bf16_bits_to_float(src[static_cast<int64_t>(r) * cols + c + e]) : 0.f;
  }
}

// ---------------------------------------------------------------------------------------------- normalise
// One 64 x 64 tile of the padded, oriented X0 per iteration.  kFromUser: source is rec.W (dmuon_ns_batched),
// else rec.U (the staged U of the Muon step).
template <typename T, bool kFromUser>
__global__ void __launch_bounds__(kThreads) normalize_kernel(const MatRec* __restrict__ recs,
                                                             const int64_t* __restrict__ prefix, int count,
                                                             int64_t total_tiles, const float* __restrict__ inv_norm) {
  __shared__ float tile[kTile][kTile + 1];
  const int tr = threadIdx.x >> 3;          // 0..31
  const int tc = (threadIdx.x & 7) * 8;     // 0, 8, .., 56
  for (int64_t t = blockIdx.x; t < total_tiles; t += gridDim.x) {
    const int mat = find_matrix(prefix, count, t);
    const MatRec& rec = recs[mat];
    const int64_t local = t - __ldg(prefix + mat);
    const int tiles_j = rec.n_pad / kTile;
    const int ti = static_cast<int>(local / tiles_j), tj = static_cast<int>(local % tiles_j);
    const uint16_t* __restrict__ src = static_cast<const uint16_t*>(kFromUser ? rec.W : rec.U);
    T* __restrict__ dst = static_cast<T*>(rec.X0);
    const float inv = __ldg(inv_norm + mat);
    const bool vec_ok = (rec.cols & 7) == 0;
    if (!rec.transposed) {
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int i = ti * kTile + tr + 32 * h, j = tj * kTile + tc;
        float f[8];
        load8_bf16_guarded(src, rec.rows, rec.cols, i, j, vec_ok, f);
#pragma unroll
        for (int e = 0; e < 8; ++e) f[e] *= inv;
        Store8<T>::run(dst + static_cast<int64_t>(i) * rec.n_pad + j, f);
      }
    } else {
      // X[i][j] = src[j][i]: stage the source tile (stored rows j, stored cols i) and read it transposed
      __syncthreads();
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int sj = tj * kTile + tr + 32 * h, si = ti * kTile + tc;
        float f[8];
        load8_bf16_guarded(src, rec.rows, rec.cols, sj, si, vec_ok, f);
#pragma unroll
        for (int e = 0; e < 8; ++e) tile[tr + 32 * h][tc + e] = f[e] * inv;
      }
      __syncthreads();
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int il = tr + 32 * h;
        float f[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) f[e] = tile[tc + e][il];
        Store8<T>::run(dst + static_cast<int64_t>(ti * kTile + il) * rec.n_pad + tj * kTile + tc, f);
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------- a6 / NS output
// One 64 x 64 tile of the STORED orientation per iteration.  kApply: W' = W - lr (scale O + wd W); else out = bf16(O).
template <typename T, bool kApply>
__global__ void __launch_bounds__(kThreads) apply_kernel(const MatRec* __restrict__ recs,
                                                         const int64_t* __restrict__ prefix, int count,
                                                         int64_t total_tiles, float lr, float wd) {
  __shared__ float tile[kTile][kTile + 1];
  const int tr = threadIdx.x >> 3;
  const int tc = (threadIdx.x & 7) * 8;
  for (int64_t t = blockIdx.x; t < total_tiles; t += gridDim.x) {
    const int mat = find_matrix(prefix, count, t);
    const MatRec& rec = recs[mat];
    const int64_t local = t - __ldg(prefix + mat);
    const int tiles_c = (rec.cols + kTile - 1) / kTile;
    const int tR = static_cast<int>(local / tiles_c), tC = static_cast<int>(local % tiles_c);
    const T* __restrict__ O = static_cast<const T*>(rec.O);
    uint16_t* __restrict__ W = static_cast<uint16_t*>(rec.W);
    const bool vec_ok = (rec.cols & 7) == 0;
    const float s_o = lr * rec.scale;
    if (rec.transposed) {
      // O(R, C) = Obuf[C][R]: stage Obuf rows [tC*64, +64), cols [tR*64, +64)  (always inside the padded buffer)
      __syncthreads();
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        float f[8];
        Load8<T>::run(O + static_cast<int64_t>(tC * kTile + tr + 32 * h) * rec.n_pad + tR * kTile + tc, f);
#pragma unroll
        for (int e = 0; e < 8; ++e) tile[tr + 32 * h][tc + e] = f[e];
      }
      __syncthreads();
    }
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int R = tR * kTile + tr + 32 * h, C = tC * kTile + tc;
      if (R >= rec.rows || C >= rec.cols) continue;
      float o[8];
      if (rec.transposed) {
#pragma unroll
        for (int e = 0; e < 8; ++e) o[e] = tile[tc + e][tr + 32 * h];
      } else {
        Load8<T>::run(O + static_cast<int64_t>(R) * rec.n_pad + C, o);
      }
      uint16_t* wp = W + static_cast<int64_t>(R) * rec.cols + C;
      if (kApply && rec.W32 != nullptr) {
        // fp32 master weights: the update is applied to the master, W is its bf16 rounding
        float* mp = rec.W32 + static_cast<int64_t>(R) * rec.cols + C;
        for (int e = 0; e < 8 && C + e < rec.cols; ++e) {
          const float w0 = mp[e];
          const float w1 = w0 - fmaf(s_o, o[e], lr * wd * w0);
          mp[e] = w1;
          wp[e] = static_cast<uint16_t>(float_to_bf16_bits(w1));
        }
      } else if (vec_ok && C + 8 <= rec.cols) {
        float w[8];
        if (kApply) {
          unpack8(*reinterpret_cast<const uint4*>(wp), w);
#pragma unroll
          for (int e = 0; e < 8; ++e) w[e] = w[e] - fmaf(s_o, o[e], lr * wd * w[e]);
        } else {
#pragma unroll
          for (int e = 0; e < 8; ++e) w[e] = o[e];
        }
        *reinterpret_cast<uint4*>(wp) = pack8_bf16(w);
      } else {
        for (int e = 0; e < 8 && C + e < rec.cols; ++e) {
          float w = o[e];
          if (kApply) {
            const float w0 = bf16_bits_to_float(wp[e]);
            w = w0 - fmaf(s_o, o[e], lr * wd * w0);
          }
          wp[e] = static_cast<uint16_t>(float_to_bf16_bits(w));
        }
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------- fast paths
// Path A (matrix not transposed, rows and cols multiples of 128, fp16 workspace): the workspace buffer has the stored
// layout, so normalise and apply are flat streaming passes: 4 x 16-byte loads per thread in flight, two elements per
// arithmetic instruction (f32x2), one 16-byte store per 8 elements.
__device__ __forceinline__ uint32_t float2_to_half2_bits(float2 f) {
  const __half2 h = __float22half2_rn(f);
  return *reinterpret_cast<const uint32_t*>(&h);
}
__device__ __forceinline__ float2 half2_bits_to_float2(uint32_t w) {
  return __half22float2(*reinterpret_cast<const __half2*>(&w));
}
// one 32-bit word (two elements) of the update  W' = W - (lr scale O + lr wd W), rounded once to bf16
__device__ __forceinline__ uint32_t apply_word(uint32_t w_bits, uint32_t o_bits, float2 so2, float2 lrwd2) {
  const float2 w = bf16x2_to_float2(w_bits);
  const float2 o = half2_bits_to_float2(o_bits);
  const float2 t = __ffma2_rn(so2, o, __fmul2_rn(lrwd2, w));
  return float2_to_bf16x2(__ffma2_rn(make_float2(-1.f, -1.f), t, w));      // w - t, one rounding
}

// 8 consecutive elements with fp32 master weights: the update is applied to the master in fp32, the
// bf16 parameter is the rounding of the new master.  o4: 8 fp16 values of O; mp: 8 floats of the master (32-byte aligned).
__device__ __forceinline__ uint4 apply8_master(float* __restrict__ mp, const uint4& o4, float2 so2, float2 lrwd2) {
  const float4 m0 = *reinterpret_cast<const float4*>(mp), m1 = *reinterpret_cast<const float4*>(mp + 4);
  const float2 w[4] = {make_float2(m0.x, m0.y), make_float2(m0.z, m0.w), make_float2(m1.x, m1.y), make_float2(m1.z, m1.w)};
  const uint32_t ow[4] = {o4.x, o4.y, o4.z, o4.w};
  float2 n[4];
  uint32_t r[4];
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    const float2 t = __ffma2_rn(so2, half2_bits_to_float2(ow[e]), __fmul2_rn(lrwd2, w[e]));
    n[e] = __ffma2_rn(make_float2(-1.f, -1.f), t, w[e]);
    r[e] = float2_to_bf16x2(n[e]);
  }
  *reinterpret_cast<float4*>(mp) = make_float4(n[0].x, n[0].y, n[1].x, n[1].y);
  *reinterpret_cast<float4*>(mp + 4) = make_float4(n[2].x, n[2].y, n[3].x, n[3].y);
  return make_uint4(r[0], r[1], r[2], r[3]);
}

template <bool kFromUser>
__global__ void __launch_bounds__(kThreads) normalize_flat_kernel(const MatRec* __restrict__ recs,
                                                                  const int64_t* __restrict__ prefix, int count,
                                                                  int64_t total_chunks,
                                                                  const float* __restrict__ inv_norm) {
  constexpr int kIter = kFlatChunk / (kThreads * 8);
  for (int64_t chunk = blockIdx.x; chunk < total_chunks; chunk += gridDim.x) {
    const int mat = find_matrix(prefix, count, chunk);
    const MatRec& rec = recs[mat];
    const int64_t start = (chunk - __ldg(prefix + mat)) * kFlatChunk;
    const uint16_t* __restrict__ src = static_cast<const uint16_t*>(kFromUser ? rec.W : rec.U) + start;
    uint16_t* __restrict__ dst = static_cast<uint16_t*>(rec.X0) + start;
    const float inv = __ldg(inv_norm + mat);
    const float2 inv2 = make_float2(inv, inv);
    uint4 v[kIter];
#pragma unroll
    for (int it = 0; it < kIter; ++it) v[it] = __ldcs(reinterpret_cast<const uint4*>(src + (it * kThreads + threadIdx.x) * 8));
#pragma unroll
    for (int it = 0; it < kIter; ++it) {
      const uint32_t w[4] = {v[it].x, v[it].y, v[it].z, v[it].w};
      uint32_t o[4];
#pragma unroll
      for (int e = 0; e < 4; ++e) o[e] = float2_to_half2_bits(__fmul2_rn(bf16x2_to_float2(w[e]), inv2));
      *reinterpret_cast<uint4*>(dst + (it * kThreads + threadIdx.x) * 8) = make_uint4(o[0], o[1], o[2], o[3]);
    }
  }
}

template <bool kApply, bool kMaster>
__global__ void __launch_bounds__(kThreads) apply_flat_kernel(const MatRec* __restrict__ recs,
                                                              const int64_t* __restrict__ prefix, int count,
                                                              int64_t total_chunks, float lr, float wd) {
  constexpr int kIter = kFlatChunk / (kThreads * 8);
  for (int64_t chunk = blockIdx.x; chunk < total_chunks; chunk += gridDim.x) {
    const int mat = find_matrix(prefix, count, chunk);
    const MatRec& rec = recs[mat];
    const int64_t start = (chunk - __ldg(prefix + mat)) * kFlatChunk;
    const uint16_t* __restrict__ O = static_cast<const uint16_t*>(rec.O) + start;
    uint16_t* __restrict__ W = static_cast<uint16_t*>(rec.W) + start;
    const float so = lr * rec.scale, lrwd = lr * wd;
    const float2 so2 = make_float2(so, so), lrwd2 = make_float2(lrwd, lrwd);
    uint4 o4[kIter], w4[kIter];
    if (kMaster) {
      float* __restrict__ M32 = rec.W32 + start;
#pragma unroll
      for (int it = 0; it < kIter; ++it) o4[it] = __ldcs(reinterpret_cast<const uint4*>(O + (it * kThreads + threadIdx.x) * 8));
#pragma unroll
      for (int it = 0; it < kIter; ++it) {
        const int off = (it * kThreads + threadIdx.x) * 8;
        *reinterpret_cast<uint4*>(W + off) = apply8_master(M32 + off, o4[it], so2, lrwd2);
      }
      continue;
    }
#pragma unroll
    for (int it = 0; it < kIter; ++it) {
      const int off = (it * kThreads + threadIdx.x) * 8;
      o4[it] = __ldcs(reinterpret_cast<const uint4*>(O + off));
      if (kApply) w4[it] = __ldcs(reinterpret_cast<const uint4*>(W + off));
    }
#pragma unroll
    for (int it = 0; it < kIter; ++it) {
      const uint32_t ow[4] = {o4[it].x, o4[it].y, o4[it].z, o4[it].w};
      const uint32_t ww[4] = {w4[it].x, w4[it].y, w4[it].z, w4[it].w};
      uint32_t r[4];
#pragma unroll
      for (int e = 0; e < 4; ++e)
        r[e] = kApply ? apply_word(ww[e], ow[e], so2, lrwd2) : float2_to_bf16x2(half2_bits_to_float2(ow[e]));
      *reinterpret_cast<uint4*>(W + (it * kThreads + threadIdx.x) * 8) = make_uint4(r[0], r[1], r[2], r[3]);
    }
  }
}

// Path B (matrix transposed, rows and cols multiples of 128, fp16 workspace): 64 x 64 tiles transposed as raw 16-bit
// elements.  Thread (a, b) = (tid / 8, tid % 8) loads the source rows 2a, 2a+1, columns 8b .. 8b+7 (two 16-byte
// loads), pairs the two rows column by column with PRMT into 32-bit words (src[2a][c], src[2a+1][c]) and stores word
// a of transposed row c; then thread (c', k') reads 16 bytes = transposed row c', elements 8k' .. 8k'+7.  The 16-byte
// chunks of a transposed row (128 B) are XOR-swizzled with (c & 7) ^ (c >> 3) so that both the word stores and the
// 16-byte loads are free of bank conflicts.
__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t sel) {
  uint32_t r;
  asm("prmt.b32 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(sel));
  return r;
}
__device__ __forceinline__ void transpose_tile16(const uint16_t* __restrict__ src, int64_t ld, uint32_t* tile,
                                                 uint4 (&out)[2]) {
  const int a = threadIdx.x >> 3, b = threadIdx.x & 7;
  const uint4 r0 = __ldcs(reinterpret_cast<const uint4*>(src + static_cast<int64_t>(2 * a) * ld + 8 * b));
  const uint4 r1 = __ldcs(reinterpret_cast<const uint4*>(src + static_cast<int64_t>(2 * a + 1) * ld + 8 * b));
  const uint32_t w0[4] = {r0.x, r0.y, r0.z, r0.w}, w1[4] = {r1.x, r1.y, r1.z, r1.w};
  __syncthreads();                                   // the previous tile has been read out
#pragma unroll
  for (int w = 0; w < 4; ++w) {
#pragma unroll
    for (int odd = 0; odd < 2; ++odd) {
      const int c = 8 * b + 2 * w + odd;             // transposed row = source column
      const int chunk = (a >> 2) ^ (c & 7) ^ (c >> 3);
      tile[c * 32 + chunk * 4 + (a & 3)] = prmt(w0[w], w1[w], odd ? 0x7632u : 0x5410u);
    }
  }
  __syncthreads();
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    const int c = a + 32 * h, k = b;
    const int chunk = k ^ (c & 7) ^ ((c >> 3) & 7);
    out[h] = *reinterpret_cast<const uint4*>(tile + c * 32 + chunk * 4);
  }
}

template <bool kFromUser>
__global__ void __launch_bounds__(kThreads) normalize_tr_kernel(const MatRec* __restrict__ recs,
                                                                const int64_t* __restrict__ prefix, int count,
                                                                int64_t total_tiles, const float* __restrict__ inv_norm) {
  __shared__ __align__(16) uint32_t tile[kTile * 32];
  for (int64_t t = blockIdx.x; t < total_tiles; t += gridDim.x) {
    const int mat = find_matrix(prefix, count, t);
    const MatRec& rec = recs[mat];
    const int64_t local = t - __ldg(prefix + mat);
    const int tiles_c = rec.cols / kTile;
    const int tR = static_cast<int>(local / tiles_c), tC = static_cast<int>(local % tiles_c);
    const uint16_t* __restrict__ src = static_cast<const uint16_t*>(kFromUser ? rec.W : rec.U);
    uint16_t* __restrict__ dst = static_cast<uint16_t*>(rec.X0);
    const float inv = __ldg(inv_norm + mat);
    const float2 inv2 = make_float2(inv, inv);
    uint4 v[2];
    transpose_tile16(src + static_cast<int64_t>(tR) * kTile * rec.cols + tC * kTile, rec.cols, tile, v);
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const uint32_t w[4] = {v[h].x, v[h].y, v[h].z, v[h].w};
      uint32_t o[4];
#pragma unroll
      for (int e = 0; e < 4; ++e) o[e] = float2_to_half2_bits(__fmul2_rn(bf16x2_to_float2(w[e]), inv2));
      // X0[i][j] = src[j][i]: oriented row = stored column, leading dimension n_pad (= rows)
      const int64_t i = tC * kTile + (threadIdx.x >> 3) + 32 * h, j = tR * kTile + (threadIdx.x & 7) * 8;
      *reinterpret_cast<uint4*>(dst + i * rec.n_pad + j) = make_uint4(o[0], o[1], o[2], o[3]);
    }
  }
}

template <bool kApply, bool kMaster>
__global__ void __launch_bounds__(kThreads) apply_tr_kernel(const MatRec* __restrict__ recs,
                                                            const int64_t* __restrict__ prefix, int count,
                                                            int64_t total_tiles, float lr, float wd) {
  __shared__ __align__(16) uint32_t tile[kTile * 32];
  for (int64_t t = blockIdx.x; t < total_tiles; t += gridDim.x) {
    const int mat = find_matrix(prefix, count, t);
    const MatRec& rec = recs[mat];
    const int64_t local = t - __ldg(prefix + mat);
    const int tiles_c = rec.cols / kTile;
    const int tR = static_cast<int>(local / tiles_c), tC = static_cast<int>(local % tiles_c);
    const uint16_t* __restrict__ O = static_cast<const uint16_t*>(rec.O);
    uint16_t* __restrict__ W = static_cast<uint16_t*>(rec.W);
    const float so = lr * rec.scale, lrwd = lr * wd;
    const float2 so2 = make_float2(so, so), lrwd2 = make_float2(lrwd, lrwd);
    // O(R, C) = Obuf[C][R]: the source tile is Obuf rows tC*64.., columns tR*64.. (leading dimension n_pad = rows)
    uint4 w4[2];
    constexpr bool master = kMaster;
    if (kApply && !master) {
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int64_t R = tR * kTile + (threadIdx.x >> 3) + 32 * h, C = tC * kTile + (threadIdx.x & 7) * 8;
        w4[h] = __ldcs(reinterpret_cast<const uint4*>(W + R * rec.cols + C));
      }
    }
    uint4 v[2];
    transpose_tile16(O + static_cast<int64_t>(tC) * kTile * rec.n_pad + tR * kTile, rec.n_pad, tile, v);
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int64_t R = tR * kTile + (threadIdx.x >> 3) + 32 * h, C = tC * kTile + (threadIdx.x & 7) * 8;
      if (master) {
        *reinterpret_cast<uint4*>(W + R * rec.cols + C) = apply8_master(rec.W32 + R * rec.cols + C, v[h], so2, lrwd2);
        continue;
      }
      const uint32_t ow[4] = {v[h].x, v[h].y, v[h].z, v[h].w};
      const uint32_t ww[4] = {w4[h].x, w4[h].y, w4[h].z, w4[h].w};
      uint32_t r[4];
#pragma unroll
      for (int e = 0; e < 4; ++e)
        r[e] = kApply ? apply_word(ww[e], ow[e], so2, lrwd2) : float2_to_bf16x2(half2_bits_to_float2(ow[e]));
      *reinterpret_cast<uint4*>(W + R * rec.cols + C) = make_uint4(r[0], r[1], r[2], r[3]);
    }
  }
}

// Pseudo-random fp16 values in (-0.025, 0.025) for the autotuner's scratch operands (all-zero operands would draw
// far less power than real data and skew the comparison between tile configurations).
__global__ void fill_scratch_kernel(uint32_t* __restrict__ p, size_t words) {
  for (size_t i = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x; i < words;
       i += static_cast<size_t>(gridDim.x) * blockDim.x) {
    uint32_t h = static_cast<uint32_t>(i) * 2654435761u;
    h ^= h >> 15; h *= 2246822519u; h ^= h >> 13;
    const float a = (static_cast<float>(h & 0xFFFFu) - 32768.f) * (0.025f / 32768.f);
    const float b = (static_cast<float>(h >> 16) - 32768.f) * (0.025f / 32768.f);
    __half2 v = __floats2half2_rn(a, b);
    p[i] = *reinterpret_cast<uint32_t*>(&v);
  }
}

// Test hook: copy one matrix's NS result out of the internal (oriented, padded) buffer as fp32, stored orientation.
template <typename T>
__global__ void export_kernel(const T* __restrict__ O, float* __restrict__ out, int rows, int cols, int n_pad,
                              int transposed) {
  const int64_t total = static_cast<int64_t>(rows) * cols;
  for (int64_t i = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x; i < total;
       i += static_cast<int64_t>(gridDim.x) * blockDim.x) {
    const int r = static_cast<int>(i / cols), c = static_cast<int>(i % cols);
    const int64_t src = transposed ? static_cast<int64_t>(c) * n_pad + r : static_cast<int64_t>(r) * n_pad + c;
    out[i] = static_cast<float>(O[src]);
  }
}

int grid_for(int64_t work, int per_sm) {
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int64_t cap = static_cast<int64_t>(sms) * per_sm;
  return static_cast<int>(work < cap ? work : cap);
}

}  // namespace

int launch_fill_scratch(void* ptr, size_t bytes, cudaStream_t s) {
  const size_t words = bytes / 4;
  if (words == 0) return DMUON_OK;
  fill_scratch_kernel<<<grid_for(static_cast<int64_t>((words + 255) / 256), 16), 256, 0, s>>>(static_cast<uint32_t*>(ptr), words);
  DMUON_CUDA_CHECK(cudaGetLastError());
  return DMUON_OK;
}

int launch_export(const void* O, float* out, int rows, int cols, int n_pad, bool transposed, bool fp32_internal,
                  cudaStream_t s) {
  const int64_t total = static_cast<int64_t>(rows) * cols;
  const int grid = grid_for((total + 255) / 256, 16);
  if (fp32_internal) export_kernel<float><<<grid, 256, 0, s>>>(static_cast<const float*>(O), out, rows, cols, n_pad, transposed);
  else export_kernel<__half><<<grid, 256, 0, s>>>(static_cast<const __half*>(O), out, rows, cols, n_pad, transposed);
  DMUON_CUDA_CHECK(cudaGetLastError());
  return DMUON_OK;
}

int launch_momentum(const ElemTables& T, float mu, cudaStream_t s) {
  if (T.flat_chunks == 0) return DMUON_OK;
  ProfScope ps("momentum_nesterov_sumsq", s);
  flat_kernel<true><<<grid_for(T.flat_chunks, 8), kThreads, 0, s>>>(T.recs, T.flat_prefix, T.count, T.flat_chunks, mu,
                                                                    T.partials);
  DMUON_CUDA_CHECK(cudaGetLastError());
  return DMUON_OK;
}

int launch_sumsq(const ElemTables& T, cudaStream_t s) {
  if (T.flat_chunks == 0) return DMUON_OK;
  ProfScope ps("sumsq", s);
  flat_kernel<false><<<grid_for(T.flat_chunks, 8), kThreads, 0, s>>>(T.recs, T.flat_prefix, T.count, T.flat_chunks, 0.f,
                                                                     T.partials);
  DMUON_CUDA_CHECK(cudaGetLastError());
  return DMUON_OK;
}

int launch_finalize_norms(const ElemTables& T, float eps, cudaStream_t s) {
  if (T.count == 0) return DMUON_OK;
  ProfScope ps("finalize_norms", s);
  finalize_norms_kernel<<<T.count, kThreads, 0, s>>>(T.flat_prefix, T.partials, eps, T.inv_norm);
  DMUON_CUDA_CHECK(cudaGetLastError());
  return DMUON_OK;
}

int launch_normalize(const ElemTables& T, bool from_user, bool fp32_internal, cudaStream_t s) {
  if (T.ptiles + T.fa_chunks + T.fb_tiles == 0) return DMUON_OK;
  if (T.fa_chunks > 0) {
    ProfScope ps("normalize_orient_cast", s);
    const int g = grid_for(T.fa_chunks, 8);
    if (from_user) normalize_flat_kernel<true><<<g, kThreads, 0, s>>>(T.recs, T.fa_prefix, T.count, T.fa_chunks, T.inv_norm);
    else normalize_flat_kernel<false><<<g, kThreads, 0, s>>>(T.recs, T.fa_prefix, T.count, T.fa_chunks, T.inv_norm);
  }
  if (T.fb_tiles > 0) {
    ProfScope ps("normalize_orient_cast", s);
    const int g = grid_for(T.fb_tiles, 8);
    if (from_user) normalize_tr_kernel<true><<<g, kThreads, 0, s>>>(T.recs, T.fb_prefix, T.count, T.fb_tiles, T.inv_norm);
    else normalize_tr_kernel<false><<<g, kThreads, 0, s>>>(T.recs, T.fb_prefix, T.count, T.fb_tiles, T.inv_norm);
  }
  DMUON_CUDA_CHECK(cudaGetLastError());
  if (T.ptiles == 0) return DMUON_OK;
  ProfScope ps("normalize_orient_cast", s);
  const int grid = grid_for(T.ptiles, 16);
#define DMUON_NORM(TT, FU) \
  normalize_kernel<TT, FU><<<grid, kThreads, 0, s>>>(T.recs, T.ptile_prefix, T.count, T.ptiles, T.inv_norm)
  if (fp32_internal) { if (from_user) DMUON_NORM(float, true); else DMUON_NORM(float, false); }
  else               { if (from_user) DMUON_NORM(__half, true); else DMUON_NORM(__half, false); }
#undef DMUON_NORM
  DMUON_CUDA_CHECK(cudaGetLastError());
  return DMUON_OK;
}

int launch_apply(const ElemTables& T, float lr, float wd, bool fp32_internal, bool master, cudaStream_t s) {
  if (T.tiles + T.fa_chunks + T.fb_tiles == 0) return DMUON_OK;
  if (T.fa_chunks > 0) {
    ProfScope ps("apply_update", s);
    if (master) apply_flat_kernel<true, true><<<grid_for(T.fa_chunks, 8), kThreads, 0, s>>>(T.recs, T.fa_prefix, T.count, T.fa_chunks, lr, wd);
    else apply_flat_kernel<true, false><<<grid_for(T.fa_chunks, 8), kThreads, 0, s>>>(T.recs, T.fa_prefix, T.count, T.fa_chunks, lr, wd);
  }
  if (T.fb_tiles > 0) {
    ProfScope ps("apply_update", s);
    if (master) apply_tr_kernel<true, true><<<grid_for(T.fb_tiles, 8), kThreads, 0, s>>>(T.recs, T.fb_prefix, T.count, T.fb_tiles, lr, wd);
    else apply_tr_kernel<true, false><<<grid_for(T.fb_tiles, 8), kThreads, 0, s>>>(T.recs, T.fb_prefix, T.count, T.fb_tiles, lr, wd);
  }
  DMUON_CUDA_CHECK(cudaGetLastError());
  if (T.tiles == 0) return DMUON_OK;
  ProfScope ps("apply_update", s);
  const int grid = grid_for(T.tiles, 16);
  if (fp32_internal) apply_kernel<float, true><<<grid, kThreads, 0, s>>>(T.recs, T.tile_prefix, T.count, T.tiles, lr, wd);
  else               apply_kernel<__half, true><<<grid, kThreads, 0, s>>>(T.recs, T.tile_prefix, T.count, T.tiles, lr, wd);
  DMUON_CUDA_CHECK(cudaGetLastError());
  return DMUON_OK;
}

int launch_store_ns(const ElemTables& T, bool fp32_internal, cudaStream_t s) {
  if (T.tiles + T.fa_chunks + T.fb_tiles == 0) return DMUON_OK;
  if (T.fa_chunks > 0) {
    ProfScope ps("store_ns_output", s);
    apply_flat_kernel<false, false><<<grid_for(T.fa_chunks, 8), kThreads, 0, s>>>(T.recs, T.fa_prefix, T.count, T.fa_chunks, 0.f, 0.f);
  }
  if (T.fb_tiles > 0) {
    ProfScope ps("store_ns_output", s);
    apply_tr_kernel<false, false><<<grid_for(T.fb_tiles, 8), kThreads, 0, s>>>(T.recs, T.fb_prefix, T.count, T.fb_tiles, 0.f, 0.f);
  }
  DMUON_CUDA_CHECK(cudaGetLastError());
  if (T.tiles == 0) return DMUON_OK;
  ProfScope ps("store_ns_output", s);
  const int grid = grid_for(T.tiles, 16);
  if (fp32_internal) apply_kernel<float, false><<<grid, kThreads, 0, s>>>(T.recs, T.tile_prefix, T.count, T.tiles, 0.f, 0.f);
  else               apply_kernel<__half, false><<<grid, kThreads, 0, s>>>(T.recs, T.tile_prefix, T.count, T.tiles, 0.f, 0.f);
  DMUON_CUDA_CHECK(cudaGetLastError());
  return DMUON_OK;
}

}  // namespace dmuon
