// pmc_gamma_static.cu — pmc_gamma_index_static: the 3-D gamma index of pmc_gamma_index (DESIGN.md
// Reading R10) for callers that must not allocate device memory.
//
// Who that is.  pmc_gamma_index keeps its working memory (the list of lattice offsets inside the search sphere, two
// 64-bit voxel counts and the maximum of the reference grid) in buffers it obtains from cudaMalloc, or from the
// allocator given to pmc_create_with_allocator, the first time it needs them and whenever the list grows.  Some users of
// a dose-comparison call cannot live with that:
//   * a plan-optimisation or QA loop running beside a framework that has already claimed the whole of the GPU's memory
//     for its own pool: cudaMalloc then fails although the job needs only a few kilobytes;
//   * a loop with a latency budget: cudaMalloc and cudaFree may wait for all outstanding work on the device, so a call
//     that usually takes a millisecond now and then takes as long as whatever else is running;
//   * code under a "no allocation after start-up" rule (long-running services that want their memory footprint fixed
//     once the start-up phase is over).
// For them the working memory is the file-scope array below.  It is part of the library's image: every GPU that loads
// libpmc holds its PMC_GAMMA_STATIC_SCRATCH_BYTES (about 96 KB) from the moment the module is loaded until the process
// exits, whether or not this entry point is ever called.
//
// This file is a translation unit of its own.  The array, the one-time look-up of its device address and the launches
// that use it must live together, and nothing of the existing pmc_gamma_index path is touched.  The kernels are copies
// of pmc_gamma.cuh's with the three scratch pointers replaced by one pointer to the Scratch block.
#include "../../include/pmc.h"

#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>
#include <cmath>
#include <cstddef>
#include <cstdio>
#include <mutex>

#include "pmc_ctx_access.h"

namespace {

constexpr int MAX_OFF = PMC_GAMMA_STATIC_MAX_OFFSETS;
constexpr int MAX_DEVICES = 64;

struct Offset { int16_t i, j, k, pad; float d2_over_dta2; };          // 12 bytes, sorted by distance
struct Scratch {
  // --- the part every call must find zeroed (HEAD_BYTES, cleared on the stream before the first kernel)
  unsigned long long n_eval, n_pass;    // voxels at or above the dose threshold; those with gamma <= 1
  uint32_t dmax_bits;                   // bit pattern of max(D_ref) (non-negative floats order like unsigned integers)
  uint32_t pad[59];
  // --- the part every call overwrites as far as it reads it
  Offset off[MAX_OFF];
};
constexpr size_t HEAD_BYTES = 256;
static_assert(offsetof(Scratch, off) == HEAD_BYTES, "head of the scratch block is 256 bytes");
static_assert(sizeof(Scratch) == PMC_GAMMA_STATIC_SCRATCH_BYTES, "pmc.h states the size of the scratch block");

// The scratch itself.  In HOST code `g_scratch` is only a handle for the runtime's symbol calls: it is not a device
// address, and handing it to a kernel would make the kernel read and write whatever host or unmapped memory the
// handle's value happens to name.  Host code therefore goes through scratch_of() below.
static __device__ __align__(256) unsigned char g_scratch[sizeof(Scratch)];

// Everything below the entry point's argument checks runs under this lock, up to and including the wait for the stream:
// one array per GPU means one call in flight per GPU, and the host-side staging array is shared as well.
std::mutex g_lock;
Scratch *g_dev_ptr[MAX_DEVICES] = {};          // device address of g_scratch on each device, looked up once
struct Keyed { double d2; int seq; Offset f; };
Keyed g_stage[MAX_OFF];                        // host staging of the offset list (static: no heap, no large stack frame)
Offset g_sorted[MAX_OFF];

// Device address of this device's copy of g_scratch.  `device` must be the current device: the runtime answers for the
// current device's instance of the symbol.  Called with g_lock held.
cudaError_t scratch_of(int device, Scratch **out) {
  if (!g_dev_ptr[device]) {
    void *p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_scratch);
    if (e != cudaSuccess) return e;
    g_dev_ptr[device] = static_cast<Scratch *>(p);
  }
  *out = g_dev_ptr[device];
  return cudaSuccess;
}

__global__ void __launch_bounds__(256) gamma_max_static_kernel(const float *ref, uint32_t n, Scratch *S) {
  float m = 0.f;
  for (uint32_t v = blockIdx.x * blockDim.x + threadIdx.x; v < n; v += gridDim.x * blockDim.x) m = fmaxf(m, ref[v]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0 && m > 0.f) atomicMax(&S->dmax_bits, __float_as_uint(m));
}

// One thread per reference voxel; offsets are visited nearest first, so the search ends as soon as the distance term
// alone reaches the best value so far (same arithmetic, in the same order, as pmc::gamma_kernel).
__global__ void __launch_bounds__(256) gamma_static_kernel(const float *__restrict__ ref, const float *__restrict__ ev, int nx, int ny,
                                                           int nz, int n_off, float inv_dd_frac, float low_dose_frac,
                                                           float *__restrict__ out, Scratch *S) {
  const float dmax = __uint_as_float(S->dmax_bits);
  const float inv_dd = dmax > 0.f ? inv_dd_frac / dmax : 0.f, thr = low_dose_frac * dmax;
  const Offset *__restrict__ off = S->off;
  const int x = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y * blockDim.y + threadIdx.y, z = blockIdx.z;
  unsigned long long n_eval = 0, n_pass = 0;
  if (x < nx && y < ny) {
    const size_t v = ((size_t)z * ny + y) * nx + x;
    const float dr = ref[v];
    float g = -1.0f;
    if (dmax > 0.f && dr >= thr) {
      float best = 3.0e38f;
      for (int o = 0; o < n_off; ++o) {
        const Offset f = off[o];
        if (f.d2_over_dta2 >= best) break;
        const int xx = x + f.i, yy = y + f.j, zz = z + f.k;
        if (xx < 0 || xx >= nx || yy < 0 || yy >= ny || zz < 0 || zz >= nz) continue;
        const float d = (__ldg(ev + ((size_t)zz * ny + yy) * nx + xx) - dr) * inv_dd;
        best = fminf(best, f.d2_over_dta2 + d * d);
      }
      g = sqrtf(best);
      n_eval = 1; n_pass = g <= 1.0f ? 1 : 0;
    }
    out[v] = g;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { n_eval += __shfl_xor_sync(0xffffffffu, n_eval, o); n_pass += __shfl_xor_sync(0xffffffffu, n_pass, o); }
  if (((threadIdx.y * blockDim.x + threadIdx.x) & 31) == 0 && n_eval) { atomicAdd(&S->n_eval, n_eval); atomicAdd(&S->n_pass, n_pass); }
}

int cuda_fail(pmc_ctx *c, cudaError_t e, const char *where) {
  char b[256]; snprintf(b, sizeof b, "pmc_gamma_index_static: %s: %s", where, cudaGetErrorString(e));
  return pmc::ctx_fail(c, PMC_E_CUDA, b);
}
#define CKS(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return cuda_fail(c, e__, #call); } while (0)

}  // namespace

extern "C" int pmc_gamma_index_static(pmc_ctx *c, const float *ref_dev, const float *eval_dev, int nx, int ny, int nz, double dx,
                                      double dy, double dz, double dd_frac, double dta_cm, double low_dose_frac, double search_cm,
                                      float *gamma_dev, double *pass_rate_host) {
  if (!c || !ref_dev || !eval_dev || !gamma_dev) return pmc::ctx_fail(c, PMC_E_INVALID_ARG, "null argument");
  if (nx < 1 || ny < 1 || nz < 1 || !(dx > 0) || !(dy > 0) || !(dz > 0) || (double)nx * ny * nz >= 2147483648.0)
    return pmc::ctx_fail(c, PMC_E_INVALID_ARG, "bad grid");
  if (!(dd_frac > 0) || !(dta_cm > 0) || !(low_dose_frac >= 0)) return pmc::ctx_fail(c, PMC_E_INVALID_ARG, "criteria must be positive");
  if (nz > 65535) return pmc::ctx_fail(c, PMC_E_UNSUPPORTED, "nz > 65535");
  if (!(search_cm > 0)) search_cm = 2.0 * dta_cm;
  const int device = pmc::ctx_device(c);
  if (device < 0 || device >= MAX_DEVICES) return pmc::ctx_fail(c, PMC_E_UNSUPPORTED, "pmc_gamma_index_static: device ordinal above 63");
  const int rx = (int)std::floor(search_cm / dx + 1e-9), ry = (int)std::floor(search_cm / dy + 1e-9), rz = (int)std::floor(search_cm / dz + 1e-9);
  if (rx > 32767 || ry > 32767 || rz > 32767 || (double)(2 * rx + 1) * (2 * ry + 1) * (2 * rz + 1) > 4.0e6)
    return pmc::ctx_fail(c, PMC_E_CAPACITY, "pmc_gamma_index_static: the search sphere holds more voxel offsets than the fixed scratch "
                                            "(PMC_GAMMA_STATIC_MAX_OFFSETS = 8192); shrink search_cm or use pmc_gamma_index");

  std::lock_guard<std::mutex> hold(g_lock);
  // lattice offsets inside the search sphere in the enumeration order of pmc_gamma_index, then nearest first with the
  // enumeration order deciding between equal distances (what its stable sort does)
  int n_off = 0;
  for (int k = -rz; k <= rz; ++k) for (int j = -ry; j <= ry; ++j) for (int i = -rx; i <= rx; ++i) {
    const double d2 = (i * dx) * (i * dx) + (j * dy) * (j * dy) + (k * dz) * (k * dz);
    if (d2 > search_cm * search_cm * (1 + 1e-12)) continue;
    if (n_off == MAX_OFF) {
      char b[256];
      snprintf(b, sizeof b, "pmc_gamma_index_static: more than %d voxel offsets within %.4g cm of a voxel: beyond the fixed scratch; "
                            "shrink search_cm or use pmc_gamma_index", MAX_OFF, search_cm);
      return pmc::ctx_fail(c, PMC_E_CAPACITY, b);
    }
    Keyed &q = g_stage[n_off];
    q.d2 = d2; q.seq = n_off; q.f.i = (int16_t)i; q.f.j = (int16_t)j; q.f.k = (int16_t)k; q.f.pad = 0; q.f.d2_over_dta2 = (float)(d2 / (dta_cm * dta_cm));
    ++n_off;
  }
  std::sort(g_stage, g_stage + n_off, [](const Keyed &a, const Keyed &b) { return a.d2 < b.d2 || (a.d2 == b.d2 && a.seq < b.seq); });   // in place
  for (int i = 0; i < n_off; ++i) g_sorted[i] = g_stage[i].f;

  CKS(cudaSetDevice(device));
  Scratch *S = nullptr;
  CKS(scratch_of(device, &S));
  cudaStream_t s = pmc::ctx_stream(c);
  CKS(cudaMemsetAsync(S, 0, HEAD_BYTES, s));                      // the previous call's counts and maximum
  CKS(cudaMemcpyAsync(S->off, g_sorted, (size_t)n_off * sizeof(Offset), cudaMemcpyHostToDevice, s));   // S->off: address arithmetic only
  const uint32_t nvox = (uint32_t)((size_t)nx * ny * nz);
  gamma_max_static_kernel<<<pmc::ctx_sm_count(c) * 8, 256, 0, s>>>(ref_dev, nvox, S);
  const dim3 blk(32, 8, 1), grd((nx + 31) / 32, (ny + 7) / 8, nz);
  gamma_static_kernel<<<grd, blk, 0, s>>>(ref_dev, eval_dev, nx, ny, nz, n_off, (float)(1.0 / dd_frac), (float)low_dose_frac, gamma_dev, S);
  unsigned long long cnt[2] = {0, 0};
  CKS(cudaMemcpyAsync(cnt, S, sizeof(cnt), cudaMemcpyDeviceToHost, s));
  CKS(cudaStreamSynchronize(s));
  CKS(cudaGetLastError());
  if (pass_rate_host) *pass_rate_host = cnt[0] ? (double)cnt[1] / (double)cnt[0] : 1.0;
  return PMC_OK;
}
