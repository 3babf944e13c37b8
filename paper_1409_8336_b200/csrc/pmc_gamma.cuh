// pmc_gamma.cuh — 3-D gamma index between two dose grids ("3D gamma index ... also computed on the
// GPU", ref [34]; Low et al.; DESIGN.md Reading R10).  One thread per reference voxel; the lattice offsets inside the
// search radius are visited in order of increasing distance, so the search stops as soon as the distance term alone
// reaches the best value found (the remaining offsets cannot lower the minimum).  A warp covers 32 consecutive x, so
// every offset is one coalesced 128-byte read of the evaluated grid that the L1/L2 serve many times over.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace pmc {

struct GammaOffset { int16_t i, j, k, pad; float d2_over_dta2; };     // sorted by d2
struct GammaParams {
  int nx, ny, nz, n_off;
  float inv_dd_frac;        // 1 / dd_frac: dose term is ((De - Dr) / (dd_frac * Dmax))^2
  float low_dose_frac;
};

// max of a non-negative float grid: the bit pattern of a non-negative float orders like an unsigned integer
__global__ void __launch_bounds__(256) gamma_max_kernel(const float *ref, uint32_t n, uint32_t *dmax_bits) {
  float m = 0.f;
  for (uint32_t v = blockIdx.x * blockDim.x + threadIdx.x; v < n; v += gridDim.x * blockDim.x) m = fmaxf(m, ref[v]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0 && m > 0.f) atomicMax(dmax_bits, __float_as_uint(m));
}

__global__ void __launch_bounds__(256) gamma_kernel(const float *__restrict__ ref, const float *__restrict__ ev,
                                                    const GammaOffset *__restrict__ off, GammaParams G,
                                                    const uint32_t *dmax_bits, float *__restrict__ out,
                                                    unsigned long long *counts /* [0] evaluated, [1] gamma <= 1 */) {
  const float dmax = __uint_as_float(*dmax_bits);
  const float inv_dd = dmax > 0.f ? G.inv_dd_frac / dmax : 0.f, thr = G.low_dose_frac * dmax;
  const int x = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y * blockDim.y + threadIdx.y, z = blockIdx.z;
  unsigned long long n_eval = 0, n_pass = 0;
  if (x < G.nx && y < G.ny) {
    const size_t v = ((size_t)z * G.ny + y) * G.nx + x;
    const float dr = ref[v];
    float g = -1.0f;
    if (dmax > 0.f && dr >= thr) {
      float best = 3.0e38f;
      for (int o = 0; o < G.n_off; ++o) {
        const GammaOffset f = off[o];
        if (f.d2_over_dta2 >= best) break;                      // sorted by distance: nothing closer is left
        const int xx = x + f.i, yy = y + f.j, zz = z + f.k;
        if (xx < 0 || xx >= G.nx || yy < 0 || yy >= G.ny || zz < 0 || zz >= G.nz) continue;
        const float d = (__ldg(ev + ((size_t)zz * G.ny + yy) * G.nx + xx) - dr) * inv_dd;
        best = fminf(best, f.d2_over_dta2 + d * d);
      }
      g = sqrtf(best);
      n_eval = 1; n_pass = g <= 1.0f ? 1 : 0;
    }
    out[v] = g;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { n_eval += __shfl_xor_sync(0xffffffffu, n_eval, o); n_pass += __shfl_xor_sync(0xffffffffu, n_pass, o); }
  if (((threadIdx.y * blockDim.x + threadIdx.x) & 31) == 0 && n_eval) { atomicAdd(counts, n_eval); atomicAdd(counts + 1, n_pass); }
}

}  // namespace pmc
