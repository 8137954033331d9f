// mg_pipes.cuh -- FP64 pipe microbenchmarks behind mg_measure_fp64_pipes (include/mg5b200.h).
//
// SURVEY.md section 7 ("microbenchmark DMMA-only, DFMA-only and interleaved before committing") and 8(d) ("measure the
// sustained DFMA ... peaks ... and DMMA m8n8k4 likewise"): the colour sum J^dagger C J for
// ncolor = 120 is a (64 x 120) x (120 x 120) real contraction per work item (64 rows = 32 helicity lanes x {re, im}).
// Whether it belongs on the FP64 tensor path (legacy mma.sync m8n8k4, tcgen05 has no f64 kind) depends on whether DMMA
// runs beside the plain DFMA pipe or on it, which these kernels measure:
//   mode 0  DFMA only, register chains            mode 1  DMMA only, register chains
//   mode 2  both, interleaved in every warp       mode 3  both, even warps DFMA / odd warps DMMA
//   mode 4  DMMA fed from shared memory in the layout of the jamp tile (A: 64 rows x K = 120, B: colour-matrix fragments)
//   mode 5  DFMA colour form fed from shared memory (one jamp element + 8 broadcast matrix elements per 16 DFMA)
// One CTA of 512 threads per SM, as the amplitude kernel of g g -> t t~ g g g runs.
#pragma once
#include <cuda_runtime.h>

__device__ __forceinline__ void mg_dmma(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

enum { MG_PIPES_DFMA_PER_BODY = 32, MG_PIPES_DMMA_PER_BODY = 4, MG_PIPES_K = 120 };

template <int MODE> __global__ void __launch_bounds__(512, 1) mg_pipes_kernel(double* out, int iters, double a, double b) {
  extern __shared__ __align__(16) double pipes_smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double x[8], c[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) { x[k] = (double)(threadIdx.x + k); c[k] = 0.0; }
  const bool do_fma = MODE == 0 || MODE == 2 || (MODE == 3 && !(warp & 1));
  const bool do_mma = MODE == 1 || MODE == 2 || (MODE == 3 && (warp & 1));
  if (MODE <= 3) {
    const double fa = 1.0 + 1e-9 * lane, fb = 1.0 - 1e-9 * lane;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        if (do_fma) {
#pragma unroll
          for (int k = 0; k < 8; ++k) x[k] = fma(x[k], a, b);
        }
        if (do_mma) mg_dmma(c[2 * u], c[2 * u + 1], fa, fb);
      }
    }
  } else if (MODE == 4) {
    // shared memory: X[K][64] (flow-major jamp tile, halves of every 16-double group swapped for odd flows so that the
    // four k of an A fragment fall into distinct bank groups), then the colour matrix as B fragments [15*15 blocks][2][32]
    double* X = pipes_smem;
    double* Bf = pipes_smem + MG_PIPES_K * 64;
    for (int i = threadIdx.x; i < MG_PIPES_K * 64 + 225 * 64; i += blockDim.x) pipes_smem[i] = 1e-3 * (i % 97);
    __syncthreads();
    // warp: m-tile pair (2 x 8 rows) x n-block pair, register tile of 4 accumulators; per k-step 2 A + 2 B loads, 4 DMMA
    const int mt = (warp & 3) * 2, r = lane >> 2, kq = lane & 3;
    for (int it = 0; it < iters; ++it) {
      for (int nb = (warp >> 2); nb < 15; nb += 8) {
        for (int kb = 0; kb < 15; ++kb) {
#pragma unroll
          for (int ks = 0; ks < 2; ++ks) {
            const int k = kb * 8 + ks * 4 + kq;
            const double a0 = X[k * 64 + ((mt * 8 + r) ^ ((k & 1) << 3))], a1 = X[k * 64 + (((mt + 1) * 8 + r) ^ ((k & 1) << 3))];
            const double b0 = Bf[((kb * 15 + nb) * 2 + ks) * 32 + lane], b1 = Bf[((kb * 15 + (nb + 4 < 15 ? nb + 4 : nb)) * 2 + ks) * 32 + lane];
            mg_dmma(c[0], c[1], a0, b0); mg_dmma(c[2], c[3], a0, b1); mg_dmma(c[4], c[5], a1, b0); mg_dmma(c[6], c[7], a1, b1);
          }
        }
      }
    }
  } else {
    // the DFMA form of the colour stage: thread = (row group of 8 rows, helicity lane); per column one (re, im) jamp element
    // and 8 broadcast matrix elements feed 16 DFMA
    double* X = pipes_smem;
    double* Cs = pipes_smem + MG_PIPES_K * 64;
    for (int i = threadIdx.x; i < MG_PIPES_K * 64 + MG_PIPES_K * MG_PIPES_K; i += blockDim.x) pipes_smem[i] = 1e-3 * (i % 97);
    __syncthreads();
    const double2* X2 = reinterpret_cast<const double2*>(X);
    for (int it = 0; it < iters; ++it) {
      const double* Cg = Cs + (warp % 15) * 8 * MG_PIPES_K;
#pragma unroll 4
      for (int t = 0; t < MG_PIPES_K; ++t) {
        const double2 j = X2[t * 32 + lane];
        const double2* cr = reinterpret_cast<const double2*>(Cg + t * 8);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const double2 cc = cr[q];
          x[2 * q] = fma(cc.x, j.x, x[2 * q]); c[2 * q] = fma(cc.x, j.y, c[2 * q]);
          x[2 * q + 1] = fma(cc.y, j.x, x[2 * q + 1]); c[2 * q + 1] = fma(cc.y, j.y, c[2 * q + 1]);
        }
      }
    }
  }
  double s = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += x[k] + c[k];
  if (s == 123456789.0) out[0] = s;
}

// flops one CTA executes per iteration, split into (plain FMA, tensor)
static void mg_pipes_flops(int mode, double* fma_flops, double* mma_flops) {
  const double warps = 16;
  const double f = 2.0 * 32 * MG_PIPES_DFMA_PER_BODY, m = 512.0 * MG_PIPES_DMMA_PER_BODY;
  *fma_flops = *mma_flops = 0;
  switch (mode) {
    case 0: *fma_flops = warps * f; break;
    case 1: *mma_flops = warps * m; break;
    case 2: *fma_flops = warps * f; *mma_flops = warps * m; break;
    case 3: *fma_flops = warps / 2 * f; *mma_flops = warps / 2 * m; break;
    case 4: {                             // warps 0..7 walk n-blocks {0, 8}, warps 8..15 {1, 9}, ... : count per warp
      double n = 0;
      for (int w = 0; w < 16; ++w) for (int nb = w >> 2; nb < 15; nb += 8) n += 15 * 2 * 4;
      *mma_flops = n * 512.0;
    } break;
    default: *fma_flops = warps * 32 * MG_PIPES_K * 16 * 2.0; break;
  }
}
