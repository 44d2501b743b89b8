// HBM-bound kernels of the Muon step (DESIGN.md steps a1, a2, a6 and the orientation/normalisation pass):
//
//   momentum_kernel   M' = mu M + G ; U = bf16(G + mu M') ; per-chunk sum of squares of the rounded U   (a1 + a2)
//   sumsq_kernel      per-chunk sum of squares of a bf16 matrix                                          (a2 alone)
//   finalize_norms    1 / (||U||_F + eps) per matrix, fixed-order (deterministic) second reduction stage
//   normalize_kernel  X0 = U / (||U||_F + eps), transposed when rows > cols, zero padded to the
//                     128-multiples the GEMM tiles want, cast to the internal dtype (fp16, or fp32 in check mode)
//   apply_kernel      W' = W - lr (scale O + wd W)  (a6; Eq. 1)  /  out = bf16(O) for dmuon_ns_batched
//
//   adamw_kernel      decoupled AdamW for the non-matrix parameters (Alg. 1 l.16)
//
// All global accesses are 128-bit and coalesced on the fast path (cols % 8 == 0); other shapes take a scalar path.
// Work is cut into fixed-size chunks/tiles over all matrices of a bucket, so one launch covers the whole bucket.
// Aligned matrices (rows and cols multiples of 128) keep the stored layout in the workspace -- tall ones included,
// the GEMM family has products for both orientations -- so their passes are flat streams; for them a6 and the NS
// output are fused into the last X-update epilogue (gemm_sm100.cu) and the kernels here run only when steps = 0.
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
// double -> bf16 with ONE rounding (RNE): round to odd at binary32 (truncate, set the last bit when inexact; binary32
// carries 16 more bits than bf16, so no tie of the second rounding can be created or lost), then RNE to bf16.
__device__ __forceinline__ uint32_t double_to_bf16_bits(double x) {
  float f = __double2float_rz(x);
  if (static_cast<double>(f) != x) f = __uint_as_float(__float_as_uint(f) | 1u);
  return float_to_bf16_bits(f);
}

// kMomentum: read G, M; write M' (in place) and U; accumulate |bf16(U)|^2.   !kMomentum: accumulate |X|^2 of rec.W.
// kExact (check mode): M' and U are formed in binary64 and rounded once, i.e. the two quantisation decisions are taken
// exactly as the fp64 oracle takes them; the fast path forms them in binary32 (one fused rounding each), which lands
// on the neighbouring bf16 value for the ~1.5 % of elements whose exact value sits within 2^-24 of a bf16 tie.
template <bool kMomentum, bool kExact>
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
            if (kExact) {
              const double mud = static_cast<double>(mu);
              const double mnx = mud * static_cast<double>(mf.x) + static_cast<double>(gf.x);     // M' = mu M + G
              const double mny = mud * static_cast<double>(mf.y) + static_cast<double>(gf.y);
              const double ux = static_cast<double>(gf.x) + mud * mnx;                            // U = G + mu M'
              const double uy = static_cast<double>(gf.y) + mud * mny;
              mo[e] = double_to_bf16_bits(mnx) | (double_to_bf16_bits(mny) << 16);
              uo[e] = double_to_bf16_bits(ux) | (double_to_bf16_bits(uy) << 16);
            } else {
              const float2 mn = __ffma2_rn(mu2, mf, gf);            // M' = mu M + G
              const float2 uf = __ffma2_rn(mu2, mn, gf);            // U  = G + mu M'   (from the unrounded M')
              mo[e] = float2_to_bf16x2(mn);
              uo[e] = float2_to_bf16x2(uf);
            }
            const float2 ur = bf16x2_to_float2(uo[e]);            // the rounded U is what the norm is taken of
            acc2 = __ffma2_rn(ur, ur, acc2);
          }
          *reinterpret_cast<uint4*>(M + i) = make_uint4(mo[0], mo[1], mo[2], mo[3]);
          *reinterpret_cast<uint4*>(U + i) = make_uint4(uo[0], uo[1], uo[2], uo[3]);
        } else {
          for (int64_t j = i; j < end; ++j) {       // ragged tail of the matrix
            const float g = bf16_bits_to_float(G[j]), m = bf16_bits_to_float(M[j]);
            uint32_t ub, mb;
            if (kExact) {
              const double mud = static_cast<double>(mu);
              const double mn = mud * static_cast<double>(m) + static_cast<double>(g);
              mb = double_to_bf16_bits(mn);
              ub = double_to_bf16_bits(static_cast<double>(g) + mud * mn);
            } else {
              const float mn = fmaf(mu, m, g);
              mb = float_to_bf16_bits(mn);
              ub = float_to_bf16_bits(fmaf(mu, mn, g));
            }
            M[j] = static_cast<uint16_t>(mb);
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
__global__ void __launch_bounds__(kThreads) finalize_norms_kernel(const MatRec* __restrict__ recs,
                                                                  const int64_t* __restrict__ prefix,
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
  // the internal buffers hold c X0 with c = rec.xscale, a power of two (exact; keeps fp16 away from its subnormals)
  if (threadIdx.x == 0)
    inv_norm[mat] = static_cast<float>(static_cast<double>(recs[mat].xscale) / (sqrt(red[0]) + static_cast<double>(eps)));
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
    const float s_o = kApply ? lr * rec.scale * rec.inv_xscale : rec.inv_xscale;    // the buffer holds c O
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
          for (int e = 0; e < 8; ++e) w[e] = o[e] * s_o;
        }
        *reinterpret_cast<uint4*>(wp) = pack8_bf16(w);
      } else {
        for (int e = 0; e < 8 && C + e < rec.cols; ++e) {
          float w = o[e] * s_o;
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
// Aligned matrices (rows and cols multiples of 128, fp16 workspace): the workspace buffer has the stored layout, so
// normalise and (for steps = 0) apply are flat streaming passes: 4 x 16-byte loads per thread in flight, two elements per
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
    const float so = kApply ? lr * rec.scale * rec.inv_xscale : rec.inv_xscale, lrwd = lr * wd;   // the buffer holds c O
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
        r[e] = kApply ? apply_word(ww[e], ow[e], so2, lrwd2) : float2_to_bf16x2(__fmul2_rn(half2_bits_to_float2(ow[e]), so2));
      *reinterpret_cast<uint4*>(W + (it * kThreads + threadIdx.x) * 8) = make_uint4(r[0], r[1], r[2], r[3]);
    }
  }
}

// ---------------------------------------------------------------------------------------------- AdamW
// Non-matrix parameters (embeddings, norms, biases; PAPER.md:239 / Alg. 1 l.16 "non-matrix params: AdamW"): decoupled
// weight decay (the paper's citation [16]), bias-corrected moments, fp32 moments and arithmetic, bf16
// parameter rounded once (reading N17 of DESIGN.md).  One flat launch over all tensors: 24 B/element
// (read p, g, m, v; write p, m, v).
__device__ __forceinline__ float adamw_one(float p, float g, float& m, float& v, const AdamScalars& sc) {
  m = fmaf(sc.beta1, m, (1.f - sc.beta1) * g);
  v = fmaf(sc.beta2, v, (1.f - sc.beta2) * g * g);
  const float denom = fmaf(sqrtf(v), sc.inv_sqrt_bc2, sc.eps);
  const float decayed = p * (1.f - sc.lr * sc.wd);
  return decayed - (sc.lr * sc.inv_bc1) * (m / denom);
}

__global__ void __launch_bounds__(kThreads) adamw_kernel(const AdamRec* __restrict__ recs,
                                                         const int64_t* __restrict__ prefix, int count,
                                                         int64_t total_chunks, const AdamScalars sc) {
  constexpr int kIter = kFlatChunk / (kThreads * 8);
  for (int64_t chunk = blockIdx.x; chunk < total_chunks; chunk += gridDim.x) {
    const int t = find_matrix(prefix, count, chunk);
    const AdamRec rec = recs[t];
    const int64_t start = (chunk - __ldg(prefix + t)) * kFlatChunk;
    const int64_t end = min(start + static_cast<int64_t>(kFlatChunk), rec.numel);
    uint16_t* __restrict__ P = static_cast<uint16_t*>(rec.p);
    const uint16_t* __restrict__ G = static_cast<const uint16_t*>(rec.g);
    float* __restrict__ M = rec.m;
    float* __restrict__ V = rec.v;
#pragma unroll
    for (int it = 0; it < kIter; ++it) {
      const int64_t i = start + (static_cast<int64_t>(it) * kThreads + threadIdx.x) * 8;
      if (i + 8 <= end) {
        float p[8], g[8];
        unpack8(__ldcs(reinterpret_cast<const uint4*>(P + i)), p);
        unpack8(__ldcs(reinterpret_cast<const uint4*>(G + i)), g);
        const float4 m0 = __ldcs(reinterpret_cast<const float4*>(M + i)), m1 = __ldcs(reinterpret_cast<const float4*>(M + i) + 1);
        const float4 v0 = __ldcs(reinterpret_cast<const float4*>(V + i)), v1 = __ldcs(reinterpret_cast<const float4*>(V + i) + 1);
        float m[8] = {m0.x, m0.y, m0.z, m0.w, m1.x, m1.y, m1.z, m1.w};
        float v[8] = {v0.x, v0.y, v0.z, v0.w, v1.x, v1.y, v1.z, v1.w};
#pragma unroll
        for (int e = 0; e < 8; ++e) p[e] = adamw_one(p[e], g[e], m[e], v[e], sc);
        *reinterpret_cast<uint4*>(P + i) = pack8_bf16(p);
        reinterpret_cast<float4*>(M + i)[0] = make_float4(m[0], m[1], m[2], m[3]);
        reinterpret_cast<float4*>(M + i)[1] = make_float4(m[4], m[5], m[6], m[7]);
        reinterpret_cast<float4*>(V + i)[0] = make_float4(v[0], v[1], v[2], v[3]);
        reinterpret_cast<float4*>(V + i)[1] = make_float4(v[4], v[5], v[6], v[7]);
      } else {
        for (int64_t j = i; j < end; ++j) {        // ragged tail of the tensor
          float m = M[j], v = V[j];
          const float pn = adamw_one(bf16_bits_to_float(P[j]), bf16_bits_to_float(G[j]), m, v, sc);
          P[j] = static_cast<uint16_t>(float_to_bf16_bits(pn));
          M[j] = m;
          V[j] = v;
        }
      }
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
                              int transposed, float inv_xscale) {
  const int64_t total = static_cast<int64_t>(rows) * cols;
  for (int64_t i = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x; i < total;
       i += static_cast<int64_t>(gridDim.x) * blockDim.x) {
    const int r = static_cast<int>(i / cols), c = static_cast<int>(i % cols);
    const int64_t src = transposed ? static_cast<int64_t>(c) * n_pad + r : static_cast<int64_t>(r) * n_pad + c;
    out[i] = static_cast<float>(O[src]) * inv_xscale;
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
                  float inv_xscale, cudaStream_t s) {
  const int64_t total = static_cast<int64_t>(rows) * cols;
  const int grid = grid_for((total + 255) / 256, 16);
  if (fp32_internal) export_kernel<float><<<grid, 256, 0, s>>>(static_cast<const float*>(O), out, rows, cols, n_pad, transposed, inv_xscale);
  else export_kernel<__half><<<grid, 256, 0, s>>>(static_cast<const __half*>(O), out, rows, cols, n_pad, transposed, inv_xscale);
  DMUON_CUDA_CHECK(cudaGetLastError());
  return DMUON_OK;
}

int launch_momentum(const ElemTables& T, float mu, bool exact, cudaStream_t s) {
  if (T.flat_chunks == 0) return DMUON_OK;
  ProfScope ps("momentum_nesterov_sumsq", s);
  if (exact) flat_kernel<true, true><<<grid_for(T.flat_chunks, 8), kThreads, 0, s>>>(T.recs, T.flat_prefix, T.count, T.flat_chunks, mu, T.partials);
  else flat_kernel<true, false><<<grid_for(T.flat_chunks, 8), kThreads, 0, s>>>(T.recs, T.flat_prefix, T.count, T.flat_chunks, mu,
                                                                          T.partials);
  DMUON_CUDA_CHECK(cudaGetLastError());
  return DMUON_OK;
}

int launch_sumsq(const ElemTables& T, cudaStream_t s) {
  if (T.flat_chunks == 0) return DMUON_OK;
  ProfScope ps("sumsq", s);
  flat_kernel<false, false><<<grid_for(T.flat_chunks, 8), kThreads, 0, s>>>(T.recs, T.flat_prefix, T.count, T.flat_chunks, 0.f,
                                                                            T.partials);
  DMUON_CUDA_CHECK(cudaGetLastError());
  return DMUON_OK;
}

int launch_finalize_norms(const ElemTables& T, float eps, cudaStream_t s) {
  if (T.count == 0) return DMUON_OK;
  ProfScope ps("finalize_norms", s);
  finalize_norms_kernel<<<T.count, kThreads, 0, s>>>(T.recs, T.flat_prefix, T.partials, eps, T.inv_norm);
  DMUON_CUDA_CHECK(cudaGetLastError());
  return DMUON_OK;
}

int launch_normalize(const ElemTables& T, bool from_user, bool fp32_internal, cudaStream_t s) {
  if (T.ptiles + T.fa_chunks == 0) return DMUON_OK;
  if (T.fa_chunks > 0) {
    ProfScope ps("normalize_cast", s);
    const int g = grid_for(T.fa_chunks, 8);
    if (from_user) normalize_flat_kernel<true><<<g, kThreads, 0, s>>>(T.recs, T.fa_prefix, T.count, T.fa_chunks, T.inv_norm);
    else normalize_flat_kernel<false><<<g, kThreads, 0, s>>>(T.recs, T.fa_prefix, T.count, T.fa_chunks, T.inv_norm);
  }
  DMUON_CUDA_CHECK(cudaGetLastError());
  if (T.ptiles == 0) return DMUON_OK;
  ProfScope ps("normalize_cast", s);
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
  if (T.tiles + T.fa_chunks == 0) return DMUON_OK;
  if (T.fa_chunks > 0) {
    ProfScope ps("apply_update", s);
    if (master) apply_flat_kernel<true, true><<<grid_for(T.fa_chunks, 8), kThreads, 0, s>>>(T.recs, T.fa_prefix, T.count, T.fa_chunks, lr, wd);
    else apply_flat_kernel<true, false><<<grid_for(T.fa_chunks, 8), kThreads, 0, s>>>(T.recs, T.fa_prefix, T.count, T.fa_chunks, lr, wd);
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
  if (T.tiles + T.fa_chunks == 0) return DMUON_OK;
  if (T.fa_chunks > 0) {
    ProfScope ps("store_ns_output", s);
    apply_flat_kernel<false, false><<<grid_for(T.fa_chunks, 8), kThreads, 0, s>>>(T.recs, T.fa_prefix, T.count, T.fa_chunks, 0.f, 0.f);
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

int launch_adamw(const AdamRec* d_recs, const int64_t* d_prefix, int count, int64_t total_chunks, const AdamScalars& sc,
                 cudaStream_t s) {
  if (total_chunks == 0) return DMUON_OK;
  ProfScope ps("adamw_update", s);
  adamw_kernel<<<grid_for(total_chunks, 8), kThreads, 0, s>>>(d_recs, d_prefix, count, total_chunks, sc);
  DMUON_CUDA_CHECK(cudaGetLastError());
  return DMUON_OK;
}

// ---------------------------------------------------------------------------------------------- AdamW, no allocation
// dmuon_adamw_step_noalloc (include/dmuon.h).  adamw_kernel reads a work table -- one AdamRec per tensor plus the chunk
// prefix -- from global memory; dmuon_adamw_step cudaMallocs that table.  Here the table lives in device memory that
// belongs to the library image itself, so a call needs nothing from the CUDA allocator.  The array is part of every
// context that loads libdmuon (192 KiB per GPU, held until the process exits).
struct AdamStaticTable {
  AdamRec recs[kAdamStaticMaxTensors];
  int64_t prefix[kAdamStaticMaxTensors + 1];
};
static __device__ __align__(256) unsigned char g_adam_static[sizeof(AdamStaticTable)];

namespace {
// On the host the name g_adam_static is only a handle for the runtime's symbol lookup, NOT the array's device address
// (handing &g_adam_static to a kernel would make it read host memory or fault).  The real address differs per device
// and is looked up once per device below.
AdamStaticTable* g_adam_static_dev[kMaxDevices] = {};
AdamStaticTable g_adam_static_host;        // where a call assembles its table (calls are serialised by the API lock)
}  // namespace

int launch_adamw_static(void* const* params, const void* const* grads, void* const* exp_avg, void* const* exp_avg_sq,
                        const int64_t* numel, int count, const AdamScalars& sc, cudaStream_t s) {
  if (count <= 0) return DMUON_OK;
  if (count > kAdamStaticMaxTensors) {
    set_error("dmuon_adamw_step_noalloc: %d tensors in one call, the built-in table holds %d (split the list)", count,
              kAdamStaticMaxTensors);
    return DMUON_ERR_INVALID_ARG;
  }
  int dev = 0;
  DMUON_CUDA_CHECK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) { set_error("dmuon_adamw_step_noalloc: device ordinal %d is not supported", dev); return DMUON_ERR_UNSUPPORTED_DEVICE; }
  if (!g_adam_static_dev[dev]) {           // first call on this device (it is the current one): resolve the address
    void* p = nullptr;
    DMUON_CUDA_CHECK(cudaGetSymbolAddress(&p, g_adam_static));
    g_adam_static_dev[dev] = static_cast<AdamStaticTable*>(p);
  }
  AdamStaticTable* const tab = g_adam_static_dev[dev];
  AdamStaticTable& h = g_adam_static_host;
  h.prefix[0] = 0;
  for (int i = 0; i < count; ++i) {
    h.recs[i] = AdamRec{params[i], grads[i], static_cast<float*>(exp_avg[i]), static_cast<float*>(exp_avg_sq[i]), numel[i]};
    h.prefix[i + 1] = h.prefix[i] + (numel[i] + kFlatChunk - 1) / kFlatChunk;
  }
  // Every entry the kernel reads (recs[0..count), prefix[0..count]) is rewritten by these two copies, so nothing of an
  // earlier call's table is used and nothing has to be cleared.  The source is ordinary (pageable) host memory: the
  // runtime has taken its copy of it when cudaMemcpyAsync returns, and the transfer itself is ordered on `s` before
  // the kernel.
  DMUON_CUDA_CHECK(cudaMemcpyAsync(tab->recs, h.recs, sizeof(AdamRec) * count, cudaMemcpyHostToDevice, s));
  DMUON_CUDA_CHECK(cudaMemcpyAsync(tab->prefix, h.prefix, sizeof(int64_t) * (count + 1), cudaMemcpyHostToDevice, s));
  const int64_t total_chunks = h.prefix[count];
  adamw_kernel<<<grid_for(total_chunks, 8), kThreads, 0, s>>>(tab->recs, tab->prefix, count, total_chunks, sc);
  DMUON_CUDA_CHECK(cudaGetLastError());
  return DMUON_OK;
}

}  // namespace dmuon
