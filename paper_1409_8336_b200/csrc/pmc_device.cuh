// pmc_device.cuh — device-side building blocks shared by the kernels of libpmc (sm_100a).
//
// Philox4x32-10 counter-based RNG, fp32 table evaluation (range spline and its inverse, cross-section lerp),
// direction rotation, Lorentz boosts, the SoA particle queue with warp-aggregated push, and the energy-loss
// straggling sampler.  Citations: PAPER.md line + section; "Reading Rk" = DESIGN.md.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace pmc {

constexpr float MP = 938.27208816f, MN = 939.56542052f, ME = 0.51099895f;
constexpr double MP_D = 938.27208816, MN_D = 939.56542052;
constexpr float HBARC = 197.3269804f;           // MeV fm
constexpr float KBETHE = 0.307075f;             // MeV cm2/mol
constexpr float TWO_PI = 6.2831853071795865f;
constexpr int NSHELL = 15;                      // PAPER.md:L77 "15 constant density shells"
constexpr int MAX_ELEM = 8;
constexpr float BIG = 1e30f;

// ------------------------------------------------------------------ Philox4x32-10 (north_star; Reading R0)
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c.x, p1 = (uint64_t)0xCD9E8D57u * c.z;
    c = make_uint4((uint32_t)(p1 >> 32) ^ c.y ^ k.x, (uint32_t)p1, (uint32_t)(p0 >> 32) ^ c.w ^ k.y, (uint32_t)p0);
    k.x += 0x9E3779B9u; k.y += 0xBB67AE85u;
  }
  return c;
}

// The same block function with the key schedule (k + r * Weyl constants, r = 0..9) computed once on the host and passed
// as a kernel parameter: the round keys then sit in the constant bank / uniform registers and a block is exactly
// 20 IMAD.WIDE + 20 LOP3 (the schedule arithmetic above costs 18 more instructions per block in the step kernel).
struct RoundKeys { uint32_t k[20]; };
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, const RoundKeys &K) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t h0 = __umulhi(0xD2511F53u, c.x), l0 = 0xD2511F53u * c.x, h1 = __umulhi(0xCD9E8D57u, c.z), l1 = 0xCD9E8D57u * c.z;
    c = make_uint4(h1 ^ c.y ^ K.k[2 * r], l1, h0 ^ c.w ^ K.k[2 * r + 1], l0);
  }
  return c;
}
// stream of one particle with the host-computed key schedule (same counters and keys as Rng, hence the same blocks); the
// round keys are named at every call so that they stay in the constant bank instead of in per-thread registers
struct RngK {
  uint32_t h0, h1, pid, blk;
  __device__ __forceinline__ void init(uint64_t hist, uint32_t pid_, uint32_t blk_) { h0 = (uint32_t)hist; h1 = (uint32_t)(hist >> 32); pid = pid_; blk = blk_; }
  __device__ __forceinline__ uint4 next4(const RoundKeys &K) { return philox4x32_10(make_uint4(h0, h1, pid, blk++), K); }
  __device__ __forceinline__ uint32_t child_id(const RoundKeys &K, uint32_t k) const {
    return philox4x32_10(make_uint4(h0, h1, pid, 0x80000000u | blk), K).x ^ (k + 1u);
  }
};
// the pair (stream, keys) with the plain next4() interface of Rng, for code that is shared between the two
struct RngKRef {
  RngK &g; const RoundKeys &K;
  __device__ __forceinline__ uint4 next4() { return g.next4(K); }
};

// Per-particle stream: key = seed, counter = (history_lo, history_hi, particle id, block number).  Draws are
// handed out a block (4 words) at a time, so the only state that travels with a particle is `blk`.
struct Rng {
  uint2 key; uint32_t h0, h1, pid, blk;
  __device__ __forceinline__ void init(uint64_t seed, uint64_t hist, uint32_t pid_, uint32_t blk_) {
    key = make_uint2((uint32_t)seed, (uint32_t)(seed >> 32));
    h0 = (uint32_t)hist; h1 = (uint32_t)(hist >> 32); pid = pid_; blk = blk_;
  }
  __device__ __forceinline__ uint4 next4() { return philox4x32_10(make_uint4(h0, h1, pid, blk++), key); }
  // id of the k-th product of this particle's current event: a block with the top counter bit set is never a
  // draw block (blk < 2^31), so the child stream is decorrelated from every draw of the parent.
  __device__ __forceinline__ uint32_t child_id(uint32_t k) const {
    return philox4x32_10(make_uint4(h0, h1, pid, 0x80000000u | blk), key).x ^ (k + 1u);
  }
};
__device__ __forceinline__ float u01(uint32_t x) { return ((float)(x >> 8) + 0.5f) * (1.0f / 16777216.0f); }   // (0,1)
// the hot loop's uniforms: top 23 bits of a word placed in the mantissa of [1,2) (two instructions, no int-to-float
// conversion): (k + 1/2) 2^-23, k = 0 .. 2^23 - 1; and a 16-bit field: (k + 1/2) 2^-16
__device__ __forceinline__ float u23(uint32_t x) { return __uint_as_float((x >> 9) | 0x3f800000u) - (1.0f - 1.0f / 16777216.0f); }
__device__ __forceinline__ float u16f(uint32_t k16) { return fmaf((float)k16, 1.0f / 65536.0f, 0.5f / 65536.0f); }

// Fast fp32 arithmetic of the hot loops (the paper's -use_fast_math build was dosimetrically equivalent, PAPER.md:L203,
// L248): 2-ulp division, and series for log1p / expm1 / sincos of the small arguments that occur at almost every step
// (accurate to < 1e-7 relative there), with the library routine as the fallback.
__device__ __forceinline__ float fdiv(float a, float b) {      // MUFU.RCP + FMUL
  float q; asm("div.approx.ftz.f32 %0, %1, %2;" : "=f"(q) : "f"(a), "f"(b)); return q;
}
__device__ __forceinline__ float fsqrt(float a) { float q; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(q) : "f"(a)); return q; }
// single MUFU instructions (the __logf / __expf / rsqrtf forms carry a denormal guard of three more instructions each)
__device__ __forceinline__ float frcp(float a) { float q; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(q) : "f"(a)); return q; }
__device__ __forceinline__ float frsq(float a) { float q; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(q) : "f"(a)); return q; }
__device__ __forceinline__ float flg2(float a) { float q; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(q) : "f"(a)); return q; }
__device__ __forceinline__ float fex2(float a) { float q; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(q) : "f"(a)); return q; }
constexpr float LN2 = 0.69314718056f, LOG2E = 1.44269504089f;
__device__ __forceinline__ float flog(float a) { return flg2(a) * LN2; }
__device__ __forceinline__ float fexp(float a) { return fex2(a * LOG2E); }
// sin and cos of 2 pi u, u in (0,1): MUFU.SIN/COS (absolute error ~5e-7), for azimuths and Box-Muller
__device__ __forceinline__ void sincos_2pi(float u, float *s, float *c) { const float x = TWO_PI * u - 3.14159265358979f; *s = -__sinf(x); *c = -__cosf(x); }
__device__ __forceinline__ float log1p_small(float x) {          // ln(1 + x)
  if (fabsf(x) < 0.06f) return x * (1.0f + x * (-0.5f + x * ((1.0f / 3.0f) + x * (-0.25f + x * (0.2f - x * (1.0f / 6.0f))))));
  return flog(1.0f + x);                                        // |x| >= 0.06: relative error < 3e-6
}
__device__ __forceinline__ float expm1_small(float x) {          // e^x - 1
  if (fabsf(x) < 0.06f) return x * (1.0f + x * (0.5f + x * ((1.0f / 6.0f) + x * ((1.0f / 24.0f) + x * (1.0f / 120.0f)))));
  return fexp(x) - 1.0f;
}
__device__ __forceinline__ void sincos_small(float x, float *s, float *c) {
  if (fabsf(x) < 0.25f) {
    const float x2 = x * x;
    *s = x * (1.0f + x2 * ((-1.0f / 6.0f) + x2 * ((1.0f / 120.0f) - x2 * (1.0f / 5040.0f))));
    *c = 1.0f + x2 * (-0.5f + x2 * ((1.0f / 24.0f) + x2 * ((-1.0f / 720.0f) + x2 * (1.0f / 40320.0f))));
  } else { *s = __sinf(x); *c = __cosf(x); }      // |x| <= pi: absolute error 5e-7
}

// ------------------------------------------------------------------ device tables
struct MatBin {                 // one HU bin, 25 words
  float hu_lo, inv_dhu, dhu, rho_lo, drho;
  float slope;                  // drho / dhu
  // the bin's range table, resolved once on the host: abscissa of the inverse table, and the offsets (in floats from the
  // start of the step kernel's shared memory) of its ln R(ln E) knots, its ln E(ln R) knots and its Sigma/rho row
  float lnr_lo, lnr_hi, inv_hr; int off_e, off_r, off_sig;
  float wet;                    // f_m of Eq.1/Eq.2 (L55-63) for table 0, 1 for own tables
  float inv_x0, zoa;
  int table;
  float nfac[MAX_ELEM];         // N_A w_i / A_i * 1e-27 : (cm^2/g) per mb of element i
  float zs;                     // sum_i w_i Z_i (Z_i + 1) / A_i (Moliere chi_c^2, Reading R12)
};

struct Nucleus {                // PAPER.md:L77, Reading R6.1; type 0 = proton, 1 = neutron
  int Z, A, nshell;
  float rmax, coulomb;
  float rout[NSHELL], rho[2][NSHELL], pF[2][NSHELL], EF[2][NSHELL], V[2][NSHELL];
  double mass;                  // target ground-state mass
  int pauli; float const_sigma_mb;
};

struct Tables {
  int n_e, n_r, n_sr, n_elem, nbins, zdim, adim;
  float ln_emin, ln_emax, inv_dlne, e_min, e_max;
  float e_cut, highland, kappa_g, s_max;
  float lnr_lo[4], lnr_hi[4], inv_hr[4];
  float c_l2, c_e0;             // (ln E - ln_emin) inv_dlne = c_l2 log2(E) - c_e0
  int hu_lut_lo, hu_lut_n;
  int opt_strag, opt_mcs, opt_el, opt_ne;
  int mcs_model, mol_n; float mol_dth; const float *mol_c;   // Moliere: C0, C1, C2 back to back, [3][mol_n]
  const float *lnR, *lnR2;      // [n_sr][n_e]; y'' pre-multiplied by h^2/6
  const float *lnE, *lnE2;      // [n_sr][n_r]
  const float *sig_el, *sig_ne; // [n_elem][n_e] mb
  const float *sig_bin;         // [nbins][n_e] total macroscopic cross-section per unit density, cm^2/g
  const MatBin *bins;           // [nbins]
  const uint8_t *hu_lut;        // [hu_lut_n] HU -> bin
  const int2 *hu_lut2;          // [hu_lut_n] HU -> {density as float bits, bin}: one 8-byte load in the step kernel
  int lut_ends_vary;            // the first or last bin (one table entry each) has a density that depends on HU
  const Nucleus *nuc;           // [n_elem]
  const double *mass;           // [zdim][adim]
  const float *evap_k, *evap_c; // [6][zdim]
  int elem_z[MAX_ELEM], elem_a[MAX_ELEM];
};

struct Grid {                   // PAPER.md:L144 "CT geometry in global memory"
  const int16_t *hu; int nx, ny, nz; float d[3]; float vol;   // voxel volume, cm^3
  double dd[3];                 // voxel sizes as given (the sampler places the source in fp64: Reading R2 tie rule)
};

// energy-grid lookup shared by the range spline and the cross-section lerp
struct EIdx { int i; float b; };
__device__ __forceinline__ EIdx e_index(const Tables &T, float lnE) {
  float t = (lnE - T.ln_emin) * T.inv_dlne;
  int i = min(max((int)floorf(t), 0), T.n_e - 2);
  return {i, t - (float)i};
}
// natural cubic spline on uniform knots, y'' pre-scaled by h^2/6
__device__ __forceinline__ float spline_eval(const float *y, const float *y2, int i, float b) {
  const float a = 1.0f - b;
  return a * y[i] + b * y[i + 1] + ((a * a * a - a) * y2[i] + (b * b * b - b) * y2[i + 1]);
}
// the same on knots interleaved with their (pre-scaled) second derivatives: {y_i, y''_i}
__device__ __forceinline__ float spline_eval2(const float2 *t, int i, float b) {
  const float a = 1.0f - b; const float2 p = t[i], q = t[i + 1];
  return fmaf(a, p.x, b * q.x) + fmaf(fmaf(a * a, a, -a), p.y, fmaf(b * b, b, -b) * q.y);
}
__device__ __forceinline__ float ln_range(const Tables &T, const float *lnR, const float *lnR2, int tab, EIdx k) {
  return spline_eval(lnR + tab * T.n_e, lnR2 + tab * T.n_e, k.i, k.b);
}
// ln E of the inverse table at ln R = x (clamped like the forward table)
__device__ __forceinline__ float ln_energy_of(const Tables &T, const float *lnE, const float *lnE2, int tab, float x) {
  if (x <= T.lnr_lo[tab]) return T.ln_emin;
  if (x >= T.lnr_hi[tab]) return T.ln_emax;
  float t = (x - T.lnr_lo[tab]) * T.inv_hr[tab];
  int i = min(max((int)floorf(t), 0), T.n_r - 2);
  return spline_eval(lnE + tab * T.n_r, lnE2 + tab * T.n_r, i, t - (float)i);
}
__device__ __forceinline__ float lerp_tab(const float *tab, EIdx k) { return (1.0f - k.b) * tab[k.i] + k.b * tab[k.i + 1]; }

// ------------------------------------------------------------------ small vector helpers
struct V3 { float x, y, z; };
__device__ __forceinline__ V3 operator+(V3 a, V3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
__device__ __forceinline__ V3 operator-(V3 a, V3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
__device__ __forceinline__ V3 operator*(float s, V3 a) { return {s * a.x, s * a.y, s * a.z}; }
__device__ __forceinline__ float dot(V3 a, V3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
__device__ __forceinline__ V3 unit(V3 a) { float n = frsq(dot(a, a)); return {a.x * n, a.y * n, a.z * n}; }
// components (a,b,c) in the frame whose z axis is the unit vector d -> lab frame
__device__ __forceinline__ V3 to_lab(V3 d, float a, float b, float c) {
  const float s2 = d.x * d.x + d.y * d.y;
  if (s2 < 1e-14f) { const float sg = d.z >= 0.f ? 1.0f : -1.0f; return {a, sg * b, sg * c}; }
  const float is = frsq(s2), s = s2 * is;
  return {a * d.x * d.z * is - b * d.y * is + c * d.x, a * d.y * d.z * is + b * d.x * is + c * d.y, -a * s + c * d.z};
}
__device__ __forceinline__ V3 isotropic(uint32_t r0, uint32_t r1) {
  const float c = 2.0f * u01(r0) - 1.0f, s = fsqrt(fmaxf(0.f, 1.0f - c * c));
  float sp, cp; sincos_2pi(u01(r1), &sp, &cp);
  return {s * cp, s * sp, c};
}
// Lorentz transformation of (p,E) from a frame moving with velocity beta
__device__ __forceinline__ void boost(V3 beta, V3 &p, float &E) {
  const float b2 = dot(beta, beta);
  if (b2 <= 0.f) return;
  const float gam = frsq(1.0f - b2), bp = dot(beta, p);
  const float f = fdiv(gam * gam, gam + 1.0f) * bp + gam * E;      // (gam-1)/b2 = gam^2/(gam+1)
  p = p + f * beta;
  E = gam * (E + bp);
}

// ------------------------------------------------------------------ SoA particle queue (PAPER.md:L144 D1)
struct Queue {
  float *x, *y, *z, *u, *v, *w, *e;    // position is voxel-local (cm from the voxel's lower corner)
  int *vox;                            // linear voxel index
  uint32_t *hist, *pid, *blk, *aux;    // RNG stream; aux = element index (event queues) / product counter
  uint32_t *count; uint32_t cap;
};
struct Particle { V3 r, d; float e; int vox; uint32_t hist, pid, blk, aux; };

__device__ __forceinline__ Particle queue_load(const Queue &q, uint32_t i) {
  Particle p;
  p.r = {q.x[i], q.y[i], q.z[i]}; p.d = {q.u[i], q.v[i], q.w[i]}; p.e = q.e[i]; p.vox = q.vox[i];
  p.hist = q.hist[i]; p.pid = q.pid[i]; p.blk = q.blk[i]; p.aux = q.aux[i];
  return p;
}
// warp-aggregated slot allocation: the lanes that reach this point together share one atomicAdd
__device__ __forceinline__ uint32_t warp_alloc(uint32_t *counter) {
  const unsigned m = __activemask();
  const int lane = threadIdx.x & 31, leader = __ffs(m) - 1;
  uint32_t base = 0;
  if (lane == leader) base = atomicAdd(counter, (uint32_t)__popc(m));
  base = __shfl_sync(m, base, leader);
  return base + (uint32_t)__popc(m & ((1u << lane) - 1u));
}
// returns false on overflow (the caller raises the sticky overflow flag)
__device__ __forceinline__ bool queue_push(const Queue &q, const Particle &p) {
  const uint32_t i = warp_alloc(q.count);
  if (i >= q.cap) return false;
  q.x[i] = p.r.x; q.y[i] = p.r.y; q.z[i] = p.r.z; q.u[i] = p.d.x; q.v[i] = p.d.y; q.w[i] = p.d.z; q.e[i] = p.e;
  q.vox[i] = p.vox; q.hist[i] = p.hist; q.pid[i] = p.pid; q.blk[i] = p.blk; q.aux[i] = p.aux;
  return true;
}

// ------------------------------------------------------------------ global counters / ledger
struct Counters {
  unsigned long long n_steps, n_elastic, n_nonelastic, n_secondary, n_missed, n_inc_tries, n_zab_bad, n_inc_guard, n_inc_cap;
  double e_source, e_deposit, e_escape, e_neutron, e_gamma, e_q, e_air;
  unsigned int overflow, inc_max_stack, inc_max_out;
};
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ unsigned long long warp_sum(unsigned long long v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
// all 32 lanes must call
__device__ __forceinline__ void flush(double *dst, double v) { v = warp_sum(v); if ((threadIdx.x & 31) == 0 && v != 0.0) atomicAdd(dst, v); }
__device__ __forceinline__ void flush(unsigned long long *dst, unsigned long long v) { v = warp_sum(v); if ((threadIdx.x & 31) == 0 && v) atomicAdd(dst, v); }

// ------------------------------------------------------------------ straggling (Reading R4)
// Vavilov(kappa, beta^2) as its defining compound-Poisson process, shifted to the CSDA mean loss.  The collision
// spectrum xi/T^2 (1 - beta^2 T/Tmax) is split at T_c: collisions above T_c are sampled one by one (Poisson number by
// inversion, thinning for the (1 - beta^2 T/Tmax) factor).  Below T_c: the part under the oracle's own cut T_c0 is
// Gaussian (Reading R4); the collisions in [T_c0, T_c] add skewness, and the sum of both is drawn as a shifted gamma
// variate with the exact variance and third cumulant (its fourth cumulant, 3 k3^2 / 2 k2, is within 12 % of the
// exact xi T_c^3 / 3), through the Wilson-Hilferty cube of one normal deviate - monotone, and the plain Gaussian in
// the limit T_c -> T_c0.  T_c is chosen so that about MU_HARD hard collisions are expected, which keeps the lanes of
// a warp in step (MU_HARD = 1/2: the shape parameter of the gamma is then >= 8, its skewness <= 0.71).  kappa >= kappa_G: Gaussian, variance
// xi Tmax (1 - beta^2/2).
//
// Random bits.  One Philox block q of the caller's stream plus `spare`, 32 bits the caller has left over from its own
// block, serve the normal deviate (23 + 16 bits), the Poisson inversion (23 bits) and the first three hard-collision
// candidates (16 bits place a candidate on the 1/T^2 spectrum between T_c and Tmax - T_c is a sizeable fraction of Tmax,
// so 2^-16 steps of 1/T are fine - and 10 bits decide its thinning).  Only a fourth candidate (0.2 % of the steps)
// needs another block: the lanes of a warp stay together.
constexpr float MU_HARD = 0.5f;
__device__ __forceinline__ float hard_candidate(uint32_t pos16, uint32_t thin10, float itc, float ditc, float b2itmax) {
  const float ua = fmaf((float)thin10, 1.0f / 1024.0f, 0.5f / 1024.0f);
  const float t = frcp(fmaf(-u16f(pos16), ditc, itc));
  return ua < fmaf(-b2itmax, t, 1.0f) ? t : 0.f;
}
template <class Gen>
__device__ __forceinline__ float straggle(const Tables &T, Gen &g, float e_start, float mean_loss, float rhoL, float zoa, uint32_t spare) {
  if (rhoL <= 0.f || mean_loss <= 0.f) return mean_loss;
  // beta^2 gamma^2 = g2m - 1; 1/beta^2 = 1 + 1/(beta^2 gamma^2)
  const float gam = fmaf(e_start, 1.0f / MP, 1.0f), bg2 = fmaf(gam, gam, -1.0f), q = frcp(bg2), ib2 = 1.0f + q, b2 = frcp(ib2);
  const float den = fmaf(gam, 2.0f * (ME / MP), 1.0f + (ME / MP) * (ME / MP));
  const float tmax = (2.0f * ME) * bg2 * frcp(den), itmax = den * q * (0.5f / ME);
  const float xi = (0.5f * KBETHE) * zoa * rhoL * ib2;
  const uint4 r = g.next4();
  const float z = fsqrt(-2.0f * LN2 * flg2(u23(r.x))) * __cosf(TWO_PI * u16f(r.y >> 16));
  float loss;
  if (xi >= T.kappa_g * tmax) {
    loss = fmaf(fsqrt(xi * tmax * fmaf(-0.5f, b2, 1.0f)), z, mean_loss);
  } else {
    // T_c = 1 / (mu / xi + 1/Tmax) with mu hard collisions expected (twice as many when kappa > 1, the last centimetre of
    // the range, where the soft gamma would otherwise be too skewed), not below the oracle's cut T_c0 = min(1 keV, Tmax/100)
    const float itc0 = fmaxf(1e3f, 100.0f * itmax);
    const float itc = fminf(fmaf(xi > tmax ? 2.0f * MU_HARD : MU_HARD, frcp(xi), itmax), itc0), tc = frcp(itc), tc0 = frcp(itc0);
    const float ditc = itc - itmax, b2itmax = b2 * itmax;
    const float mu_c = xi * ditc;                                            // candidates (before thinning)
    const float mean_hard = xi * (LN2 * flg2(tmax * itc) - b2 * fmaf(-tc, itmax, 1.0f));
    // Poisson(mu_c) number of candidates by inversion with one uniform
    const float up = u23(r.z), p0 = fex2(-LOG2E * mu_c), p1 = p0 * mu_c, c1 = p0 + p1, p2 = 0.5f * p1 * mu_c, c2 = c1 + p2;
    const float h0 = hard_candidate(r.y & 0xFFFFu, spare & 0x3FFu, itc, ditc, b2itmax);
    const float h1 = hard_candidate(r.w >> 16, (spare >> 10) & 0x3FFu, itc, ditc, b2itmax);
    float hard = (up > p0 ? h0 : 0.f) + (up > c1 ? h1 : 0.f);
    if (up > c2) {                                                           // three or more: 1.4 % of the steps
      hard += hard_candidate(r.w & 0xFFFFu, (spare >> 20) & 0x3FFu, itc, ditc, b2itmax);
      float pk = p2 * mu_c * (1.0f / 3.0f), cdf = c2 + pk;
      int k = 3, avail = 0; uint4 w = make_uint4(0u, 0u, 0u, 0u);
      while (up > cdf && k < 64) {                                           // four or more: one more block per four
        if (avail == 0) { w = g.next4(); avail = 4; }
        const uint32_t v = w.x; w.x = w.y; w.y = w.z; w.z = w.w; --avail;
        hard += hard_candidate(v >> 16, v & 0x3FFu, itc, ditc, b2itmax);
        ++k; pk *= mu_c * frcp((float)k); cdf += pk;
      }
    }
    // soft part: k2 = xi tc (1 - b2 tc/2Tmax) of everything below tc; k3 = xi [t^2 (1/2 - b2 t/3Tmax)] from tc0 to tc
    const float x = b2itmax * tc, x0 = b2itmax * tc0;
    const float k2 = xi * tc * fmaf(-0.5f, x, 1.0f), sd = fsqrt(k2);
    const float k3 = xi * (tc * tc * fmaf(-1.0f / 3.0f, x, 0.5f) - tc0 * tc0 * fmaf(-1.0f / 3.0f, x0, 0.5f));
    float soft = sd * z;
    if (itc < itc0 && k3 > 0.f) {
      const float A = 2.0f * k2 * sd, isa = k3 * frcp(A), sa = A * frcp(k3), c9 = isa * isa * (1.0f / 9.0f);   // sa = sqrt(shape)
      const float e = fmaxf(fmaf(z * isa, 1.0f / 3.0f, -c9), -1.0f);
      soft = sd * sa * fmaf(e, fmaf(e, 3.0f + e, 3.0f), c9 * c9 * c9);       // sqrt(k2 a) [(1 + e)^3 - E(1 + e)^3]
    }
    loss = mean_loss + (hard - mean_hard) + soft;
  }
  return fminf(fmaxf(loss, 0.f), e_start);
}

// ------------------------------------------------------------------ Cugnon NN parameterisation (PAPER.md:L77 ref [20]; Reading R6)
// p in GeV/c, sigma in mb
// (below 0.8 GeV/c - every collision of a cascade started below 250 MeV - both branches are evaluated and one selected:
// the lanes of a warp sit at different momenta)
__device__ __forceinline__ float cug_sigma_pp(float p) {
  if (p < 0.8f) { const float a = 34.0f * fex2(-2.104f * flg2(p * 2.5f)); float d = p - 0.7f; d *= d; return p < 0.44f ? a : fmaf(1000.0f * d, d, 23.5f); }
  if (p < 2.0f) return fdiv(1250.0f, p + 50.0f) - 4.0f * (p - 1.3f) * (p - 1.3f);
  return fdiv(77.0f, p + 1.5f);
}
__device__ __forceinline__ float cug_sigma_np(float p) {
  if (p < 0.8f) {
    const float l = LN2 * flg2(p), a = 6.3555f * fex2(LOG2E * (-3.2481f * l - 0.377f * l * l)), q = fabsf(p - 0.95f);
    return p < 0.446f ? a : fmaf(196.0f * q * q, fsqrt(q), 33.0f);
  }
  if (p < 2.0f) return 31.0f * frsq(p);
  return fdiv(77.0f, p + 1.5f);
}
__device__ __forceinline__ float cug_b_pp(float p) {
  if (p < 2.0f) { float p2 = p * p, p4 = p2 * p2, p8 = p4 * p4; return fdiv(5.5f * p8, 7.7f + p8); }
  return 5.334f + 0.67f * (p - 2.0f);
}
__device__ __forceinline__ float cug_b_np(float p) {
  if (p < 0.225f) return 0.f;
  if (p < 0.6f) return 16.53f * (p - 0.225f);
  if (p < 1.6f) return -1.63f * p + 7.16f;
  return cug_b_pp(p);
}
__device__ __forceinline__ float cug_a_np(float p) { return p < 0.8f ? 1.0f : fdiv(0.64f, p * p); }

// |t| from exp(-B t) truncated to [0, tmax]
__device__ __forceinline__ float trunc_exp(float B, float tmax, float u) {
  if (B * tmax < 1e-6f) return u * tmax;
  return fdiv(-flog(1.0f - u * (1.0f - fexp(-B * tmax))), B);
}
// cos(theta_cm) of NN elastic scattering: dsigma/dt ~ exp(B t) (+ a exp(B u) for np).  Uses 2 uniforms.
__device__ __forceinline__ float sample_nn_cos(bool same, float p_lab_gev, float pcm_mev, uint32_t r0, uint32_t r1) {
  const float tmax = 4.0f * pcm_mev * pcm_mev * 1e-6f;
  const float B = same ? cug_b_pp(p_lab_gev) : cug_b_np(p_lab_gev);
  bool backward = false;
  if (!same) { const float a = cug_a_np(p_lab_gev); backward = u01(r0) * (1.0f + a) < a; }
  const float t = trunc_exp(B, tmax, u01(r1));
  const float c = 1.0f - fdiv(2.0f * t, tmax);
  return backward ? -c : c;
}

}  // namespace pmc
