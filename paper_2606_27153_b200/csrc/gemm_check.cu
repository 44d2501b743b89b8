// fp32-operand check mode (BASELINE.json north_star: "<= 1e-4 in an fp32-operand check mode"): the same three
// NS products as gemm_sm100.cu, on fp32 matrices with true fp32 FMA on the SIMT pipes (TF32 tensor cores would
// carry a 10-bit mantissa and miss the tolerance).  Dense, no symmetry shortcut.  Small shapes only.
#include "common.h"

namespace dmuon {
namespace {

constexpr int kT = 64;    // output tile edge
constexpr int kK = 16;    // K step

// C[i][j] = alpha * sum_k L(i,k) R(k,j) + beta * D[i][j],   L(i,k) = L[i*l_i + k*l_k],  R(k,j) = R[k*r_k + j*r_j]
__global__ void __launch_bounds__(256) check_gemm_kernel(const float* __restrict__ L, int64_t l_i, int64_t l_k,
                                                         const float* __restrict__ R, int64_t r_k, int64_t r_j,
                                                         const float* __restrict__ D, float* __restrict__ C, int M,
                                                         int N, int K, int64_t ldc, float alpha, float beta) {
  __shared__ float sL[kK][kT + 1];
  __shared__ float sR[kK][kT + 1];
  const int ty = threadIdx.x / 16, tx = threadIdx.x % 16;
  const int i0 = blockIdx.y * kT, j0 = blockIdx.x * kT;
  float acc[4][4] = {};
  for (int k0 = 0; k0 < K; k0 += kK) {
    for (int e = threadIdx.x; e < kT * kK; e += 256) {
      const int r = e / kK, k = e % kK;          // L tile: row r, k
      const int i = i0 + r, kk = k0 + k;
      sL[k][r] = (i < M && kk < K) ? L[i * l_i + kk * l_k] : 0.f;
      const int j = j0 + r;
      sR[k][r] = (j < N && kk < K) ? R[kk * r_k + j * r_j] : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < kK; ++k) {
      float a[4], b[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) { a[u] = sL[k][ty * 4 + u]; b[u] = sR[k][tx * 4 + u]; }
#pragma unroll
      for (int u = 0; u < 4; ++u)
#pragma unroll
        for (int v = 0; v < 4; ++v) acc[u][v] = fmaf(a[u], b[v], acc[u][v]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int u = 0; u < 4; ++u)
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      const int i = i0 + ty * 4 + u, j = j0 + tx * 4 + v;
      if (i < M && j < N) {
        float r = alpha * acc[u][v];
        if (D) r = fmaf(beta, D[i * ldc + j], r);
        C[i * ldc + j] = r;
      }
    }
}

}  // namespace

int launch_check_gemm(GemmOp op, const float* in0, const float* in1, float* out, int m, int n, float alpha, float beta,
                      cudaStream_t stream) {
  dim3 block(256);
  switch (op) {
    case OP_SYRK: {   // C[m x m] = alpha X X^T, X is m x n (ld n)
      ProfScope ps("check_syrk_fp32", stream);
      dim3 grid((m + kT - 1) / kT, (m + kT - 1) / kT);
      check_gemm_kernel<<<grid, block, 0, stream>>>(in0, n, 1, in0, 1, n, nullptr, out, m, m, n, m, alpha, 0.f);
      break;
    }
    case OP_SQ: {     // C = alpha A A + beta A
      ProfScope ps("check_sq_fp32", stream);
      dim3 grid((m + kT - 1) / kT, (m + kT - 1) / kT);
      check_gemm_kernel<<<grid, block, 0, stream>>>(in0, m, 1, in0, m, 1, in0, out, m, m, m, m, alpha, beta);
      break;
    }
    case OP_BX: {     // C[m x n] = alpha B X + beta X
      ProfScope ps("check_bx_fp32", stream);
      dim3 grid((n + kT - 1) / kT, (m + kT - 1) / kT);
      check_gemm_kernel<<<grid, block, 0, stream>>>(in0, m, 1, in1, n, 1, in1, out, m, n, m, n, alpha, beta);
      break;
    }
  }
  DMUON_CUDA_CHECK(cudaGetLastError());
  return DMUON_OK;
}

}  // namespace dmuon
