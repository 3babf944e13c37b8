// pmc_transport.cuh — beam-spot sampler, condensed-history step kernel, nuclear-elastic kernel and the
// batch-statistics kernels.
#pragma once
#include "pmc_device.cuh"

namespace pmc {

constexpr int SPOT_GUIDE = 4096;  // entries of the guide table of the spot CDF
struct SpotDev {                 // pmc_spot, prepared on the host (axis normalised, transverse basis built)
  double pos[3]; double ax[3], ex[3], ey[3];
  double e, sigma_e, sx, sy, divx, divy;
};

struct RunParams {
  uint64_t seed; uint64_t hist0;      // first history id of this launch
  RoundKeys rk;                       // Philox key schedule of `seed` (host-computed)
  uint32_t n;                         // histories in this launch
  // All B batches ("10 groups") are in flight at once, each scoring into its own tally grid:
  // history h (0-based within the call) belongs to batch floor(h B / n_total); tally of batch b starts at b * nvox.
  uint64_t local0, n_total;           // call-local index of this launch's first history; histories in the call
  uint32_t B, nvox;
  float b_over_n, inv_nx, inv_ny;     // B / n_total, 1 / nx, 1 / ny
  float *let_num, *let_den;           // LET_d tallies [nvox] (Reading R9) or nullptr
  // per-spot dose influence (Reading R11): roi_map[vox] = column or -1, dij[spot][column] in MeV
  const int32_t *roi_map; float *dij; uint32_t n_roi;
  int max_steps; float *dbg_out;      // pmc_first_steps: stop after max_steps, write [hist][8]
  int aggregate;                      // warp-aggregated dose atomics
  int skip_tally;                     // measurement only (option "dose_scoring" = 0): the step kernel scores nothing
};

// The queue word `aux` carries the spot index of the history in its upper 24 bits through every generation; the low
// byte is the target element (event queues) or the next product index (residual queue).
__device__ __forceinline__ uint32_t aux_spot(uint32_t a) { return a >> 8; }
__device__ __forceinline__ uint32_t aux_low(uint32_t a) { return a & 0xFFu; }
__device__ __forceinline__ uint32_t aux_with(uint32_t a, uint32_t low) { return (a & ~0xFFu) | (low & 0xFFu); }
__device__ __forceinline__ void score_influence(const RunParams &P, uint32_t aux, int vox, float e) {
  if (P.roi_map == nullptr || e == 0.f) return;
  const int32_t j = P.roi_map[vox];
  if (j >= 0) atomicAdd(P.dij + (size_t)aux_spot(aux) * P.n_roi + (uint32_t)j, e);
}

// floor(h B / n_total) * nvox without a 64-bit division: float estimate, exact correction
__device__ __forceinline__ uint32_t batch_base(const RunParams &P, uint32_t hist) {
  const uint64_t h = P.local0 + hist, hb = h * (uint64_t)P.B;
  uint32_t b = min((uint32_t)((float)h * P.b_over_n), P.B - 1u);
  while ((uint64_t)b * P.n_total > hb) --b;
  while ((uint64_t)(b + 1u) * P.n_total <= hb) ++b;
  return b * P.nvox;
}
// q = a / d, r = a % d for 0 <= a < 2^31, d >= 1 (float estimate, exact correction)
__device__ __forceinline__ void divmod(int a, int d, float inv_d, int &q, int &r) {
  q = (int)((float)a * inv_d); r = a - q * d;
  while (r < 0) { --q; r += d; }
  while (r >= d) { ++q; r -= d; }
}

// ------------------------------------------------------------------ material of a voxel
struct VoxMat { float rho, wf, inv_x0, zoa; int table, bin; };
__device__ __forceinline__ int hu_to_bin(const Tables &T, const uint8_t *lut, int hu) {
  return lut[min(max(hu - T.hu_lut_lo, 0), T.hu_lut_n - 1)];
}
__device__ __forceinline__ float bin_density(const MatBin &m, int hu) {
  const float t = fminf(fmaxf((float)hu - m.hu_lo, 0.f), m.dhu);
  return m.rho_lo + m.drho * (t * m.inv_dhu);
}

// Highland theta0 with the paper's factor; t = mass thickness / X0
__device__ __forceinline__ float highland(const Tables &T, float e, float t) {
  if (t <= 0.f) return 0.f;
  const float pc2 = e * (e + 2.0f * MP);
  return fdiv(T.highland * 13.6f * (e + MP), pc2) * fsqrt(t) * fmaxf(0.f, 1.0f + 0.038f * __logf(t));
}
// one MCS deflection: two independent projected Gaussians of width theta0 (Reading R3.4)
__device__ __forceinline__ V3 deflect(V3 d, float theta0, uint32_t r0, uint32_t r1) {
  const float th = theta0 * fsqrt(-2.0f * __logf(u01(r0)));
  float st, ct, sp, cp;
  sincos_small(th, &st, &ct); sincos_2pi(u01(r1), &sp, &cp);
  return unit(to_lab(d, st * cp, st * sp, ct));
}

// Full Moliere theory (Bethe 1953; Reading R12): space angle after mass thickness t of the voxel's mixture.
// chi_c^2 = 0.157 t zs / (p beta)^2; ln chi_a^2 = Z(Z+1)/A-weighted mean of ln{2.007e-5 Z^(2/3) [1 + 3.34 (Z alpha/beta)^2] / p^2};
// b = ln(chi_c^2 / chi_a^2) + 1 - 2 C_Euler; B - ln B = b; reduced angle x from the tabulated cumulative C0 + C1/B + C2/B^2
// (bisection, uniform in x^2 inside a bin), beyond the table from the Rutherford tail 1/(B x^2).  Returns a negative
// number when the step holds fewer than 20 collisions (outside the theory): the caller then uses Highland.
__device__ __forceinline__ float moliere_angle(const Tables &T, const MatBin &m, float e, float t, float u) {
  const float p2 = e * (e + 2.0f * MP), E = e + MP, ibeta2 = fdiv(E * E, p2), pb = fdiv(p2, E);
  if (!(t > 0.f) || !(m.zs > 0.f)) return -1.0f;
  float zl = 0.f;
#pragma unroll
  for (int i = 0; i < MAX_ELEM; ++i) {
    if (i < T.n_elem && m.nfac[i] > 0.f) {
      const float Z = (float)T.elem_z[i], za = Z * (1.0f / 137.035999f);
      const float q = m.nfac[i] * Z * (Z + 1.0f);                            // proportional to w Z (Z+1) / A
      zl += q * (__logf(2.007e-5f * (1.0f + 3.34f * za * za * ibeta2)) + (2.0f / 3.0f) * __logf(Z) - __logf(p2));
    }
  }
  const float qs = m.zs * (6.02214076e23f * 1e-27f);                          // same normalisation as q
  const float chic2 = fdiv(0.157f * m.zs * t, pb * pb), ln_omega = __logf(chic2) - fdiv(zl, qs);
  if (ln_omega < 2.99573227f) return -1.0f;                                  // ln 20
  const float b = ln_omega + (1.0f - 2.0f * 0.5772156649f);
  float B = b + __logf(b);
#pragma unroll
  for (int it = 0; it < 4; ++it) B -= fdiv(B - __logf(B) - b, 1.0f - fdiv(1.0f, B));
  const int n = T.mol_n; const float iB = fdiv(1.0f, B), iB2 = iB * iB;
  const float *c0 = T.mol_c, *c1 = T.mol_c + n, *c2 = T.mol_c + 2 * n;
  auto C = [&](int k) { return __ldg(c0 + k) + __ldg(c1 + k) * iB + __ldg(c2 + k) * iB2; };
  const float xmax = (float)(n - 1) * T.mol_dth, tail = fdiv(iB, xmax * xmax), cend = C(n - 1), total = cend + tail, U = u * total;
  float x;
  if (U >= cend) x = rsqrtf(B * fmaxf(total - U, 1e-30f));
  else {
    int lo = 0, hi = n - 1;                                                   // C(lo) <= U < C(hi)
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (C(mid) <= U) lo = mid; else hi = mid; }
    const float ca = C(lo), cb = C(hi), f = cb > ca ? fminf(fmaxf(fdiv(U - ca, cb - ca), 0.f), 1.0f) : 0.5f;
    const float x0 = (float)lo * T.mol_dth, x1 = (float)hi * T.mol_dth;
    x = fsqrt(x0 * x0 + f * (x1 * x1 - x0 * x0));
  }
  return fminf(fsqrt(chic2 * B) * x, 3.14159265f);
}
// rotate d by the polar angle th and a uniform azimuth
__device__ __forceinline__ V3 deflect_by(V3 d, float th, uint32_t r1) {
  float st, ct, sp, cp;
  sincos_small(th, &st, &ct); sincos_2pi(u01(r1), &sp, &cp);
  return unit(to_lab(d, st * cp, st * sp, ct));
}

// mean energy loss over water-equivalent path dr (g/cm2 of the table medium) from the range table
// (Eq.2): E - E(R(E) - dr), written with expm1 so that a vanishing step loses nothing.
__device__ __forceinline__ float mean_loss(const Tables &T, const float *lnE, const float *lnE2, int tab,
                                           float e, float lnEv, float lnRv, float Rg, float dr) {
  const float r1 = Rg - dr;
  float lnE1 = T.ln_emin;
  if (r1 > 0.f) lnE1 = ln_energy_of(T, lnE, lnE2, tab, lnRv + log1p_small(-fdiv(dr, Rg)));
  const float m = -e * expm1_small(lnE1 - lnEv);
  return fminf(fmaxf(m, 0.f), e);
}

// ------------------------------------------------------------------ K1: beam-spot sampler (Reading R2)
__device__ __forceinline__ double u01d(uint32_t x) { return ((double)x + 0.5) * (1.0 / 4294967296.0); }

__global__ void __launch_bounds__(256) sampler_kernel(Tables T, Grid G, const SpotDev *spots, const double *cdf, const uint32_t *guide, int nspots,
                                                     RunParams P, Queue out, Counters *cnt, float air_rho, float air_wf,
                                                     float air_inv_x0, float air_zoa, int air_table) {
  // Block-stride loop (same trip count for every thread of a block) so that a block makes ONE allocation in the
  // output queue per trip and one ledger flush per warp at the end: 3e5 same-address atomics per 1e7 histories cost
  // more than the sampling itself.
  __shared__ uint32_t s_cnt[8], s_base;
  double e_src = 0, e_esc = 0, e_air = 0; unsigned long long missed = 0;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (uint32_t i0 = blockIdx.x * blockDim.x; i0 < P.n; i0 += gridDim.x * blockDim.x) {
  const uint32_t i = i0 + threadIdx.x;
  bool push = false; Particle p{};
  if (i < P.n) {
    const uint64_t hist = P.hist0 + i;
    RngK gk; gk.init(hist, 0u, 0u);
    RngKRef g{gk, P.rk};
    uint4 r = g.next4();
    // spot ~ weight: first cdf entry >= u; guide[j] = first entry >= j / SPOT_GUIDE brackets the search to a spot or two
    const double us = u01d(r.x);
    const int gj = min((int)(us * SPOT_GUIDE), SPOT_GUIDE - 1);
    int lo = (int)guide[gj], hi = min((int)guide[gj + 1], nspots - 1);
    while (lo < hi) { int mid = (lo + hi) >> 1; if (cdf[mid] < us) lo = mid + 1; else hi = mid; }
    const SpotDev sp = spots[lo];
    // Gaussian deviates in fp32 (relative error 1e-7 of sigma), accumulated onto the fp64 spot position
    const double rr = (double)sqrtf(-2.0f * logf(u01(r.y)));
    float s2f, c2f; sincospif(2.0f * u01(r.z), &s2f, &c2f); const double s2 = s2f, c2 = c2f;
    double pos[3], dir[3];
    for (int k = 0; k < 3; ++k) { pos[k] = sp.pos[k] + sp.sx * rr * c2 * sp.ex[k] + sp.sy * rr * s2 * sp.ey[k]; dir[k] = sp.ax[k]; }
    if (sp.divx > 0 || sp.divy > 0) {
      uint4 q = g.next4();
      const double r2 = (double)sqrtf(-2.0f * logf(u01(q.x))); float s4f, c4f; sincospif(2.0f * u01(q.y), &s4f, &c4f); const double s4 = s4f, c4 = c4f;
      double n2 = 0;
      for (int k = 0; k < 3; ++k) { dir[k] = sp.ax[k] + sp.divx * r2 * c4 * sp.ex[k] + sp.divy * r2 * s4 * sp.ey[k]; n2 += dir[k] * dir[k]; }
      n2 = 1.0 / sqrt(n2); for (int k = 0; k < 3; ++k) dir[k] *= n2;
    }
    double E = sp.e;
    if (sp.sigma_e > 0) { uint4 q = g.next4(); E += sp.sigma_e * (double)(sqrtf(-2.0f * logf(u01(q.x))) * cospif(2.0f * u01(q.y))); }
    E = fmax(E, 0.0);
    e_src += E;
    const double size[3] = {G.nx * G.dd[0], G.ny * G.dd[1], G.nz * G.dd[2]};
    auto ray_box = [&](const double *o, const double *dd, double &tin) {
      double t0 = 0, t1 = 1e300;
      for (int k = 0; k < 3; ++k) {
        if (dd[k] == 0) { if (o[k] < 0 || o[k] > size[k]) return false; continue; }
        const double inv = 1.0 / dd[k];
        double ta = (0 - o[k]) * inv, tb = (size[k] - o[k]) * inv;
        if (ta > tb) { double s = ta; ta = tb; tb = s; }
        t0 = fmax(t0, ta); t1 = fmin(t1, tb);
      }
      tin = t0; return t0 < t1;
    };
    double tin; bool ok = ray_box(pos, dir, tin);
    if (!ok) { e_esc += E; missed += 1; }
    else if (tin > 0) {
      // single air step to the CT edge: hinge, Highland, mean loss + straggling
      uint4 q = g.next4();
      const double tau = u01d(q.x) * tin;
      double rh[3]; for (int k = 0; k < 3; ++k) rh[k] = pos[k] + tau * dir[k];
      double dn[3] = {dir[0], dir[1], dir[2]};
      if (T.opt_mcs) {
        V3 d1 = deflect(V3{(float)dir[0], (float)dir[1], (float)dir[2]}, highland(T, (float)E, (float)tin * air_rho * air_inv_x0), q.y, q.z);
        dn[0] = d1.x; dn[1] = d1.y; dn[2] = d1.z;
      }
      double t2;
      if (!ray_box(rh, dn, t2)) { e_esc += E; missed += 1; ok = false; }
      else {
        const double L = tau + t2;
        for (int k = 0; k < 3; ++k) { pos[k] = rh[k] + t2 * dn[k]; dir[k] = dn[k]; }
        const float ef = (float)E, lnEv = logf(fminf(fmaxf(ef, T.e_min), T.e_max));
        const float lnRv = ln_range(T, T.lnR, T.lnR2, air_table, e_index(T, lnEv)), Rg = expf(lnRv);
        float loss = mean_loss(T, T.lnE, T.lnE2, air_table, ef, lnEv, lnRv, Rg, (float)L * air_wf);
        if (T.opt_strag) loss = straggle(T, g, ef, loss, (float)L * air_rho, air_zoa, q.w);   // q.w: not used by the air step itself
        e_air += loss; E -= loss;
        if (E <= T.e_cut) { e_air += E; ok = false; }
      }
    }
    if (ok) {
      int idx[3]; const int nn[3] = {G.nx, G.ny, G.nz}; float loc[3];
      for (int k = 0; k < 3; ++k) {
        const double rv = fmin(fmax(pos[k], 0.0), size[k]), dk = G.dd[k];
        int ii = (int)floor(rv / dk);
        if (ii * dk == rv && dir[k] < 0) ii -= 1;
        ii = min(max(ii, 0), nn[k] - 1);
        idx[k] = ii; loc[k] = (float)fmin(fmax(rv - ii * dk, 0.0), dk);
      }
      p.r = {loc[0], loc[1], loc[2]}; p.d = unit(V3{(float)dir[0], (float)dir[1], (float)dir[2]}); p.e = (float)E;
      p.vox = (idx[2] * G.ny + idx[1]) * G.nx + idx[0];
      p.hist = i; p.pid = 0u; p.blk = gk.blk; p.aux = (uint32_t)lo << 8;
      push = true;
    }
  }
  // one queue allocation per block and trip
  const unsigned wm = __ballot_sync(0xffffffffu, push);
  if (lane == 0) s_cnt[wid] = (uint32_t)__popc(wm);
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t tot = 0;
    for (int k = 0; k < (int)(blockDim.x >> 5); ++k) { const uint32_t c = s_cnt[k]; s_cnt[k] = tot; tot += c; }
    s_base = tot ? atomicAdd(out.count, tot) : 0u;
  }
  __syncthreads();
  if (push) {
    const uint32_t slot = s_base + s_cnt[wid] + (uint32_t)__popc(wm & ((1u << lane) - 1u));
    if (slot < out.cap) {
      out.x[slot] = p.r.x; out.y[slot] = p.r.y; out.z[slot] = p.r.z; out.u[slot] = p.d.x; out.v[slot] = p.d.y; out.w[slot] = p.d.z;
      out.e[slot] = p.e; out.vox[slot] = p.vox; out.hist[slot] = p.hist; out.pid[slot] = p.pid; out.blk[slot] = p.blk; out.aux[slot] = p.aux;
    } else atomicOr(&cnt->overflow, 1u);
  }
  __syncthreads();
  }
  flush(&cnt->e_source, e_src); flush(&cnt->e_escape, e_esc); flush(&cnt->e_air, e_air); flush(&cnt->n_missed, missed);
}

// ------------------------------------------------------------------ dose deposit (atomics)
// Lanes of a warp that score into the same voxel in the same iteration are merged (warp match) so that a
// single RED reaches the L2; with a pencil beam the lanes advance slab by slab and collide often.
// With LET_d scoring on, the same merge also carries the step's e x LET into the numerator grid and e into the
// denominator grid (indexed by voxel, not by batch).
__device__ __forceinline__ void deposit(float *tally, uint32_t tvox, float e, bool on, int aggregate,
                                        float *let_num, float *let_den, uint32_t vox, float e_let, float let) {
  const bool has_let = let_num != nullptr;
  if (!aggregate) {
    if (on && e != 0.f) atomicAdd(tally + tvox, e);
    if (has_let && on && e_let > 0.f) { atomicAdd(let_num + vox, e_let * let); atomicAdd(let_den + vox, e_let); }
    return;
  }
  const unsigned act = __ballot_sync(0xffffffffu, on);
  if (!on) return;
  const unsigned peers = __match_any_sync(act, tvox);
  const int lane = threadIdx.x & 31, leader = __ffs(peers) - 1;
  float sum = e, sn = e_let * let, sd = e_let;
  if (peers != (1u << lane)) {
    // segmented reduction over the peer set
    sum = 0.f; sn = 0.f; sd = 0.f;
    unsigned m = peers;
    while (m) {
      const int src = __ffs(m) - 1; m &= m - 1;
      sum += __shfl_sync(peers, e, src);
      if (has_let) { sn += __shfl_sync(peers, e_let * let, src); sd += __shfl_sync(peers, e_let, src); }
    }
  }
  if (lane == leader) {
    if (sum != 0.f) atomicAdd(tally + tvox, sum);
    if (has_let && sd > 0.f) { atomicAdd(let_num + vox, sn); atomicAdd(let_den + vox, sd); }
  }
}

// ------------------------------------------------------------------ K2: condensed-history step kernel (Reading R3)
// Persistent kernel: every lane pulls a particle from the input queue, steps it in registers until it stops,
// leaves the grid or reaches a discrete nuclear event, then refills from the queue (warp-aggregated fetch).
// Particles that reach an event are appended to the elastic or non-elastic queue; nothing else is written back.
#ifndef PMC_TRANSPORT_BLOCKS
#define PMC_TRANSPORT_BLOCKS 1
#endif
#ifndef PMC_TRANSPORT_THREADS
#define PMC_TRANSPORT_THREADS 896
#endif
constexpr int TRANSPORT_THREADS = PMC_TRANSPORT_THREADS, TRANSPORT_BLOCKS_PER_SM = PMC_TRANSPORT_BLOCKS;

// distance along one axis to the face the particle is heading for (voxel-local r in [0, size], inv = 1/d); BIG if d = 0
__device__ __forceinline__ float axis_dist(float r, float d, float size) {
  const float t = fmaxf(((d > 0.f ? size : 0.f) - r) * frcp(d), 0.f);
  return d != 0.f ? t : BIG;
}
// new direction after a polar deflection (st, ct) with azimuth (sp, cp) about the unit vector d, renormalised
__device__ __forceinline__ V3 rotate(V3 d, float st, float ct, float sp, float cp) {
  const float s2 = fmaf(d.x, d.x, d.y * d.y);
  V3 n;
  if (s2 < 1e-14f) { const float sg = d.z >= 0.f ? 1.0f : -1.0f; n = {st * cp, sg * st * sp, sg * ct}; }
  else {
    const float is = frsq(s2), A = st * cp * is, B = st * sp * is, Az = A * d.z;
    n = {fmaf(Az, d.x, fmaf(-B, d.y, ct * d.x)), fmaf(Az, d.y, fmaf(B, d.x, ct * d.y)), fmaf(-A, s2, ct * d.z)};
  }
  const float in = frsq(fmaf(n.x, n.x, fmaf(n.y, n.y, n.z * n.z)));
  return {n.x * in, n.y * in, n.z * in};
}

// ---- the step kernel's tables in shared memory (PAPER.md:L144 used textures) and its look-ups, shared with step_range_kernel
// Layout from the start of the dynamic shared memory: spline knots interleaved with their second derivatives (one 8-byte
// load per knot), ln R(ln E) first, then ln E(ln R), then Sigma/rho per HU bin, the HU bins and the HU -> {density, bin}
// table; MatBin holds each bin's offsets (in floats) into these arrays.
struct StepTables { const float *f; const MatBin *bins; const int2 *lut; };
// all threads of the block call; the caller synchronises before the first look-up
__device__ __forceinline__ StepTables stage_step_tables(const Tables &T, unsigned char *smem_raw) {
  float2 *s_R = reinterpret_cast<float2 *>(smem_raw);
  float2 *s_E = s_R + T.n_sr * T.n_e;
  float *s_sig = reinterpret_cast<float *>(s_E + T.n_sr * T.n_r);
  MatBin *s_bins = reinterpret_cast<MatBin *>(s_sig + T.nbins * T.n_e);
  // 8-byte entries: the byte offset of the table is rounded up to 8 from the start of the (16-byte aligned) block - the bins
  // sit after nbins * n_e floats, i.e. at 4 mod 8 when both counts are odd, and a MatBin is 25 words.  (Offset arithmetic,
  // not pointer-to-integer casts, so that the compiler still sees a shared-memory address.)  The launch's shared-memory
  // size carries 32 spare bytes for the padding.
  const int lut_off = ((2 * T.n_sr * (T.n_e + T.n_r) + T.nbins * T.n_e) * 4 + T.nbins * (int)sizeof(MatBin) + 7) & ~7;
  int2 *s_lut = reinterpret_cast<int2 *>(smem_raw + lut_off);
  for (int i = threadIdx.x; i < T.n_sr * T.n_e; i += blockDim.x) s_R[i] = make_float2(T.lnR[i], T.lnR2[i]);
  for (int i = threadIdx.x; i < T.n_sr * T.n_r; i += blockDim.x) s_E[i] = make_float2(T.lnE[i], T.lnE2[i]);
  for (int i = threadIdx.x; i < T.nbins * T.n_e; i += blockDim.x) s_sig[i] = T.sig_bin[i];
  for (int i = threadIdx.x; i < T.nbins * (int)(sizeof(MatBin) / 4); i += blockDim.x)
    reinterpret_cast<uint32_t *>(s_bins)[i] = reinterpret_cast<const uint32_t *>(T.bins)[i];
  for (int i = threadIdx.x; i < T.hu_lut_n; i += blockDim.x) s_lut[i] = T.hu_lut2[i];
  return {reinterpret_cast<const float *>(smem_raw), s_bins, s_lut};
}
// knot and fraction of the forward tables from l2 = log2(E), E already clamped to the table: t = (ln E - ln e_min) / dlnE
// in one FMA with the two constants folded on the host
__device__ __forceinline__ EIdx step_e_index(const Tables &T, float l2) {
  const float te = fmaf(l2, T.c_l2, -T.c_e0);
  const int ke = min(max((int)te, 0), T.n_e - 2);
  return {ke, te - (float)ke};
}
// ln R (g/cm2 of the bin's table medium) at that knot position
__device__ __forceinline__ float step_ln_range(const float *s_f, const MatBin &m, EIdx k) {
  return spline_eval2(reinterpret_cast<const float2 *>(s_f + m.off_e), k.i, k.b);
}
// ln E at ln R = xr from the bin's inverse table, clamped to the table's ends
__device__ __forceinline__ float step_ln_energy(const Tables &T, const float *s_f, const MatBin &m, float xr) {
  const float tr = (xr - m.lnr_lo) * m.inv_hr;
  const int kr = min(max((int)tr, 0), T.n_r - 2);
  const float lnE1 = spline_eval2(reinterpret_cast<const float2 *>(s_f + m.off_r), kr, tr - (float)kr);
  return xr <= m.lnr_lo ? T.ln_emin : (xr >= m.lnr_hi ? T.ln_emax : lnE1);
}

// MCS_MODEL: 0 = Highland (the paper's choice), 1 = full Moliere; a template so that the default kernel carries none of
// the Moliere code or its registers
// DBG: the pmc_first_steps variant (stop after max_steps, write the state of every primary); the production kernel
// carries neither its registers nor its branches.
// EXTRA: LET_d scoring, per-spot dose influence or warp-merged dose atomics are on (the plain kernel carries none of it)
template <int MCS_MODEL, bool DBG, bool EXTRA>
__global__ void __launch_bounds__(TRANSPORT_THREADS, TRANSPORT_BLOCKS_PER_SM) transport_kernel(Tables T, Grid G, RunParams P, Queue in, uint32_t *gen_n,
                                                           uint32_t *head, Queue q_ev, float *tally, Counters *cnt) {
  // the generation's particle count stays on the device (the host does not wait for it): an empty generation ends here
  const uint32_t n_in = min(*in.count, in.cap);
  if (blockIdx.x == 0 && threadIdx.x == 0) *gen_n = n_in;
  if (n_in == 0u) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const StepTables S = stage_step_tables(T, smem_raw);
  __syncthreads();
  const float *s_f = S.f;                                         // every table offset in MatBin counts floats from here
  const MatBin *s_bins = S.bins; const int2 *s_lut = S.lut;

  const float szx = G.d[0], szy = G.d[1], szz = G.d[2];
  const int lane = threadIdx.x & 31;
  bool active = false, exhausted = false;
  Particle p; int ix = 0, iy = 0, iz = 0, nstep = 0; float path = 0.f; uint32_t tbase = 0;
  int hu = 0;                           // HU of the current voxel: fetched when the voxel changes, a step ahead of its use
  uint32_t c_steps = 0;                 // per-lane partial sums (a lane sees < 1e7 steps and < 1e4 MeV): 32-bit is enough
  float c_dep = 0.f;
  const bool nuclear = T.opt_el || T.opt_ne;

  while (true) {
    // ---- refill idle lanes (at once: waiting until several lanes are idle was measured slower, 39.4 vs 37.3 ms at 8 lanes)
    const unsigned need = __ballot_sync(0xffffffffu, !active && !exhausted);
    if (need) {
      uint32_t base = 0;
      if (lane == __ffs(need) - 1) base = atomicAdd(head, (uint32_t)__popc(need));
      base = __shfl_sync(0xffffffffu, base, __ffs(need) - 1);
      if (!active && !exhausted) {
        const uint32_t idx = base + (uint32_t)__popc(need & ((1u << lane) - 1u));
        if (idx < n_in) {
          p = queue_load(in, idx);
          int t; divmod(p.vox, G.nx, P.inv_nx, t, ix); divmod(t, G.ny, P.inv_ny, iz, iy);
          active = true; nstep = 0; path = 0.f; tbase = batch_base(P, p.hist); hu = G.hu[p.vox];
        } else exhausted = true;
      }
    }
    if (!__any_sync(0xffffffffu, active)) break;

    float dep = 0.f, let = 0.f; int dep_vox = p.vox;
    if (active) {
      // the stream is re-keyed from (history, particle, block) every step: only the block counter lives across steps
      const uint64_t hid = P.hist0 + p.hist;
      RngK gk; gk.init(hid, p.pid, p.blk);
      RngKRef g{gk, P.rk};
      // ---- material of the current voxel
      const int li = min(max(hu - T.hu_lut_lo, 0), T.hu_lut_n - 1);
      const int2 le = s_lut[li];                                  // {density of this HU, bin}
      const MatBin &m = s_bins[le.y];
      float rho = __int_as_float(le.x);
      if (T.lut_ends_vary && (li == 0 || li == T.hu_lut_n - 1)) rho = fmaf(m.slope, fminf(fmaxf((float)hu - m.hu_lo, 0.f), m.dhu), m.rho_lo);
      const float wf = rho * m.wet;
      c_steps++;
      // draws of the step: r.x nuclear distance, r.y hinge (upper half), r.z and r.w (upper half) the MCS deflection; the
      // lower halves of r.y and r.w go to the straggling sampler
      const uint4 r = g.next4();
      const uint32_t spare = __byte_perm(r.y, r.w, 0x5410);
      // ---- 1. nuclear distance, face distance, residual range
      const float e0 = p.e, l2 = flg2(fminf(fmaxf(e0, T.e_min), T.e_max)), lnEv = l2 * LN2;
      const EIdx k = step_e_index(T, l2);
      float lam = BIG;
      if (nuclear) { const float Sig = rho * lerp_tab(s_f + m.off_sig, k); lam = Sig > 0.f ? -LN2 * flg2(u23(r.x)) * frcp(Sig) : BIG; }
      const float dface = fminf(fminf(axis_dist(p.r.x, p.d.x, szx), axis_dist(p.r.y, p.d.y, szy)), axis_dist(p.r.z, p.d.z, szz));
      const float lnRv = step_ln_range(s_f, m, k), Rg = fex2(lnRv * LOG2E), iwf = frcp(wf);
      const float R = Rg * iwf, smax = T.s_max > 0.f ? T.s_max * iwf : BIG;
      // ---- 2. step = min (Reading R3.2)
      float dx = lam; int lim = 2;
      if (dface < dx) { dx = dface; lim = 1; }
      if (R < dx) { dx = R; lim = 3; }
      if (smax < dx * (1.0f - 1e-6f)) { dx = smax; lim = 0; }   // ties go to the face / event (Reading R3.2)
      // ---- 3-5. random hinge (PAPER.md:L69 ref [19]): first leg tau, deflect, second leg
      float tau = 0.f; V3 dnew = p.d;
      if (T.opt_mcs && dx > 0.f) {
        tau = u16f(r.y >> 16) * dx;
        p.r = {fmaf(tau, p.d.x, p.r.x), fmaf(tau, p.d.y, p.r.y), fmaf(tau, p.d.z, p.r.z)};
        float th = -1.0f;
        if (MCS_MODEL == 1) th = moliere_angle(T, m, e0, dx * rho, u23(r.z));
        if (th < 0.f) {
          // Highland theta0 times the Rayleigh radius of two independent projected Gaussians (Reading
          // R3.4), under one square root: theta = K (e + MP)/pc2 [1 + 0.038 ln t] sqrt(-2 t ln u)
          const float t = dx * rho * m.inv_x0;
          const float rad = fsqrt(t * (-2.0f * LN2) * flg2(u23(r.z)));
          th = (T.highland * 13.6f) * (e0 + MP) * frcp(e0 * (e0 + 2.0f * MP)) * rad * fmaxf(0.f, fmaf(0.038f * LN2, flg2(t), 1.0f));
        }
        float st, ct, sp, cp;
        sincos_small(th, &st, &ct); sincos_2pi(u16f(r.w >> 16), &sp, &cp);
        dnew = rotate(p.d, st, ct, sp, cp);
      }
      const float ell = dx - tau;
      const float tx = axis_dist(p.r.x, dnew.x, szx), ty = axis_dist(p.r.y, dnew.y, szy), tz = axis_dist(p.r.z, dnew.z, szz);
      float d2 = tx; int ax2 = 0;                                // ties: x before y before z
      if (ty < d2) { d2 = ty; ax2 = 1; }
      if (tz < d2) { d2 = tz; ax2 = 2; }
      // a face-limited step always ends on a face (dx = distance to the voxel boundary; Reading R3.5)
      const bool onface = ell >= d2 || lim == 1;
      const float leg = onface ? d2 : ell, L = tau + leg;
      const int cls = onface ? 1 : lim;
      p.r.x = fminf(fmaxf(fmaf(leg, dnew.x, p.r.x), 0.f), szx);
      p.r.y = fminf(fmaxf(fmaf(leg, dnew.y, p.r.y), 0.f), szy);
      p.r.z = fminf(fmaxf(fmaf(leg, dnew.z, p.r.z), 0.f), szz);
      p.d = dnew; if (DBG) path += L;
      // boundary step: the neighbour voxel (done before the energy loss, whose registers it would otherwise compete with;
      // if the proton stops in this step the advanced index is simply not used)
      bool exits = false;
      if (cls == 1) {                    // selects, not branches: the lanes of a warp leave through different faces
        const bool a0 = ax2 == 0, a1 = ax2 == 1;
        const bool up = (a0 ? dnew.x : a1 ? dnew.y : dnew.z) > 0.f;
        const int sg2 = up ? 1 : -1;
        ix += a0 ? sg2 : 0; iy += a1 ? sg2 : 0; iz += (a0 || a1) ? 0 : sg2;
        const float face = up ? 0.f : (a0 ? szx : a1 ? szy : szz);
        p.r.x = a0 ? face : p.r.x; p.r.y = a1 ? face : p.r.y; p.r.z = (a0 || a1) ? p.r.z : face;
        const int nidx = a0 ? ix : a1 ? iy : iz, nmax = a0 ? G.nx : a1 ? G.ny : G.nz;
        exits = (unsigned)nidx >= (unsigned)nmax;
        p.vox += sg2 * (a0 ? 1 : a1 ? G.nx : G.nx * G.ny);
        if (!exits) hu = G.hu[p.vox];
      }
      // ---- 6. energy loss from the range table (Eq.2) + straggling (L61)
      float loss;
      if (cls == 3) { loss = e0; if (EXTRA) let = L > 0.f ? fdiv(0.1f * e0, L) : 0.f; }   // 7. range-out: everything stays here (L71)
      else if (L <= 0.f) loss = 0.f;
      else {
        // E - E(R(E) - dr), written with expm1 so that a vanishing step loses nothing
        const float dr = L * wf;
        float lnE1 = T.ln_emin;
        if (Rg - dr > 0.f) {
          lnE1 = step_ln_energy(T, s_f, m, lnRv + log1p_small(-dr * frcp(Rg)));
        }
        loss = fminf(fmaxf(-e0 * expm1_small(lnE1 - lnEv), 0.f), e0);
        if (EXTRA) let = fdiv(0.1f * loss, L);                   // keV/um of this step (Reading R9)
        if (T.opt_strag) loss = straggle(T, g, e0, loss, L * rho, m.zoa, spare);
      }
      p.e = e0 - loss; dep = loss;
      bool alive = cls != 3;
      if (alive && p.e <= T.e_cut) { dep += p.e; p.e = 0.f; alive = false; }           // L71 (2)
      c_dep += dep;
      if (alive && exits) { atomicAdd(&cnt->e_escape, (double)p.e); alive = false; }   // L71 (3): leaves the grid
      if (DBG) ++nstep;
      p.blk = gk.blk;
      if (alive && cls == 2 && !DBG) {
        // ---- 8. discrete nuclear event at the end point (L71): handed to event_kernel, which picks the class and
        // the target element with all lanes busy instead of one lane of this warp
        p.vox = dep_vox;
        if (!queue_push(q_ev, p)) atomicOr(&cnt->overflow, 2u);
        alive = false;
      }
      if (DBG && alive && P.max_steps > 0 && nstep >= P.max_steps) alive = false;
      if (!alive) {
        active = false;
        if (DBG && P.dbg_out && p.pid == 0u) {
          float *o = P.dbg_out + 8ull * p.hist;
          o[0] = ix * szx + p.r.x; o[1] = iy * szy + p.r.y; o[2] = iz * szz + p.r.z;
          o[3] = p.d.x; o[4] = p.d.y; o[5] = p.d.z; o[6] = p.e; o[7] = path;
        }
      }
    }
    if (EXTRA && P.skip_tally) continue;
    if (EXTRA) {
      deposit(tally, tbase + (uint32_t)dep_vox, dep, dep != 0.f, P.aggregate, P.let_num, P.let_den, (uint32_t)dep_vox, let > 0.f ? dep : 0.f, let);
      if (P.roi_map != nullptr && dep != 0.f) score_influence(P, p.aux, dep_vox, dep);
    } else if (dep != 0.f) atomicAdd(tally + tbase + (uint32_t)dep_vox, dep);
  }
  flush(&cnt->n_steps, (unsigned long long)c_steps);
  flush(&cnt->e_deposit, (double)c_dep);
}

// ------------------------------------------------------------------ sub-step: the step kernel's own table look-ups
// R(E) and E(R) of HU bin `bin` through exactly what transport_kernel uses - the tables staged in shared memory by
// stage_step_tables, the knot index from log2(E) (step_e_index), the interleaved splines (step_ln_range, step_ln_energy)
// and the single-MUFU log2 / exp2 - so that the production look-up is compared with the oracle element by element
// (pmc_range_of_energy evaluates the global-memory splines with logf / expf / floorf instead).
__global__ void __launch_bounds__(256) step_range_kernel(Tables T, int bin, const float *in, uint64_t n, float *out, int inverse) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const StepTables S = stage_step_tables(T, smem_raw);
  __syncthreads();
  const MatBin &m = S.bins[bin];
  for (uint64_t i = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
    if (!inverse) {
      const float l2 = flg2(fminf(fmaxf(in[i], T.e_min), T.e_max));
      out[i] = fex2(step_ln_range(S.f, m, step_e_index(T, l2)) * LOG2E);
    } else out[i] = fex2(step_ln_energy(T, S.f, m, flg2(fmaxf(in[i], 1e-30f)) * LN2) * LOG2E);
  }
}

// ------------------------------------------------------------------ event class and target element (Reading R5)
// One event per thread over the event queue: elastic vs non-elastic in proportion to the macroscopic cross-sections at
// the energy after the step, then the target element in proportion to n_i sigma_i within the class.  If both vanish at
// that energy nothing happens and the proton goes on in the next generation.
__global__ void __launch_bounds__(256) event_kernel(Tables T, Grid G, RunParams P, Queue in, Queue q_el, Queue q_ne, Queue next,
                                                    Counters *cnt) {
  const uint32_t n = min(*in.count, in.cap);
  unsigned long long c_el = 0, c_ne = 0;
  for (uint32_t i0 = blockIdx.x * blockDim.x; i0 < n; i0 += gridDim.x * blockDim.x) {
    const uint32_t i = i0 + threadIdx.x;
    if (i < n) {
      Particle p = queue_load(in, i);
      Rng g; g.init(P.seed, P.hist0 + p.hist, p.pid, p.blk);
      const int hu = G.hu[p.vox];
      const MatBin &m = T.bins[hu_to_bin(T, T.hu_lut, hu)];
      const EIdx k1 = e_index(T, logf(fminf(fmaxf(p.e, T.e_min), T.e_max)));
      float pel[MAX_ELEM], pne[MAX_ELEM], sel = 0.f, sne = 0.f;
#pragma unroll
      for (int e = 0; e < MAX_ELEM; ++e) {
        pel[e] = 0.f; pne[e] = 0.f;
        if (e < T.n_elem && m.nfac[e] > 0.f) {
          if (T.opt_el) pel[e] = m.nfac[e] * lerp_tab(T.sig_el + e * T.n_e, k1);
          if (T.opt_ne) pne[e] = m.nfac[e] * lerp_tab(T.sig_ne + e * T.n_e, k1);
        }
        sel += pel[e]; sne += pne[e];
      }
      if (sel + sne > 0.f) {
        const uint4 q = g.next4();
        const bool is_el = u01(q.x) * (sel + sne) < sel;
        float u = u01(q.y) * (is_el ? sel : sne); int el = -1;
#pragma unroll
        for (int e = 0; e < MAX_ELEM; ++e) {
          const float w = is_el ? pel[e] : pne[e];
          if (w > 0.f && (el < 0 || u >= 0.f)) { el = e; u -= w; }
        }
        p.aux = aux_with(p.aux, (uint32_t)el); p.blk = g.blk;
        if (is_el) { c_el++; if (!queue_push(q_el, p)) atomicOr(&cnt->overflow, 2u); }
        else { c_ne++; if (!queue_push(q_ne, p)) atomicOr(&cnt->overflow, 4u); }
      } else if (!queue_push(next, p)) atomicOr(&cnt->overflow, 8u);
    }
  }
  flush(&cnt->n_elastic, c_el); flush(&cnt->n_nonelastic, c_ne);
}

// ------------------------------------------------------------------ nuclear elastic (Eq.3; Reading R5)
struct ElasticOut { float t_gev2, T_out, T_rec; V3 dir_out, dir_rec; };
// proton of kinetic energy Tk along +z on nucleus of mass M (MeV); r = 4 random words
__device__ __forceinline__ ElasticOut elastic_event(int A, float M, float Tk, uint4 r) {
  const float E = Tk + MP, plab = sqrtf(Tk * (Tk + 2.0f * MP));
  const float s = MP * MP + M * M + 2.0f * M * E, irs = rsqrtf(s), pcm = M * plab * irs;
  const float tmax = 4.0f * pcm * pcm * 1e-6f;
  float t;
  if (A == 1) {
    t = trunc_exp(cug_b_pp(plab * 1e-3f), tmax, u01(r.y));                  // p-p: Cugnon angular law
  } else {
    const float lA = __logf((float)A);
    float a1, b1, a2, b2 = 10.0f;
    if (A <= 62) { a1 = __expf(1.63f * lA); b1 = 14.5f * __expf(0.66f * lA); a2 = 1.4f * __expf(0.33f * lA); }
    else { a1 = __expf(1.33f * lA); b1 = 60.0f * __expf(0.33f * lA); a2 = 0.4f * __expf(0.4f * lA); }
    const float w1 = a1 * (1.0f - __expf(-b1 * tmax)) / b1, w2 = a2 * (1.0f - __expf(-b2 * tmax)) / b2;
    const float bb = u01(r.x) * (w1 + w2) < w1 ? b1 : b2;
    t = trunc_exp(bb, tmax, u01(r.y));                                      // |t|, truncated exponential
  }
  const float ct = 1.0f - 2.0f * t / tmax, st = sqrtf(fmaxf(0.f, 1.0f - ct * ct));
  float sp, cp; sincospif(2.0f * u01(r.z), &sp, &cp);
  // boost of the CM momenta along z with beta = plab/(E+M)
  const float beta = plab / (E + M), gam = rsqrtf(1.0f - beta * beta);
  const float Ep = sqrtf(pcm * pcm + MP * MP), Er = sqrtf(pcm * pcm + M * M);
  V3 po{pcm * st * cp, pcm * st * sp, gam * (pcm * ct + beta * Ep)};
  V3 pr{-po.x, -po.y, gam * (-pcm * ct + beta * Er)};
  ElasticOut o;
  o.t_gev2 = t;
  o.T_rec = t * 1e6f / (2.0f * M);            // invariant: t = -2 M T_rec, free of the E - M cancellation
  o.T_out = Tk - o.T_rec;
  o.dir_out = unit(po);
  o.dir_rec = dot(pr, pr) > 0.f ? unit(pr) : V3{0.f, 0.f, 1.f};
  return o;
}

// K-elastic: one event per thread over the elastic queue; the scattered proton (and, for hydrogen, the recoil
// proton) go to the next-generation transport queue; recoil nuclei deposit locally (L79 policy).
__global__ void __launch_bounds__(256) elastic_kernel(Tables T, RunParams P, Queue in, Queue out, float *tally, Counters *cnt) {
  const uint32_t n = min(*in.count, in.cap);
  double c_dep = 0; unsigned long long c_sec = 0;
  for (uint32_t i0 = blockIdx.x * blockDim.x; i0 < n; i0 += gridDim.x * blockDim.x) {
    const uint32_t i = i0 + threadIdx.x;
    if (i < n) {
      Particle p = queue_load(in, i);
      Rng g; g.init(P.seed, P.hist0 + p.hist, p.pid, p.blk);
      const int el = (int)aux_low(p.aux), Z = T.elem_z[el], A = T.elem_a[el];
      const float M = (float)T.mass[Z * T.adim + A];
      const ElasticOut o = elastic_event(A, M, p.e, g.next4());
      const V3 d0 = p.d;
      float dep = 0.f;
      Particle s = p;
      p.d = unit(to_lab(d0, o.dir_out.x, o.dir_out.y, o.dir_out.z)); p.e = o.T_out; p.aux = aux_with(p.aux, 0u);
      bool push_rec = false;
      if (A == 1 && o.T_rec > T.e_cut) {
        s.d = unit(to_lab(d0, o.dir_rec.x, o.dir_rec.y, o.dir_rec.z)); s.e = o.T_rec;
        s.pid = g.child_id(0u); s.blk = 0u; s.aux = aux_with(p.aux, 0u); push_rec = true; c_sec++;
      } else dep += o.T_rec;
      p.blk = g.blk;
      const bool push_p = p.e > T.e_cut;
      if (!push_p) dep += p.e;
      if (push_p) { if (!queue_push(out, p)) atomicOr(&cnt->overflow, 8u); }
      if (push_rec) { if (!queue_push(out, s)) atomicOr(&cnt->overflow, 8u); }
      if (dep != 0.f) { atomicAdd(tally + batch_base(P, p.hist) + (uint32_t)p.vox, dep); c_dep += (double)dep; score_influence(P, p.aux, p.vox, dep); }
    }
  }
  flush(&cnt->e_deposit, c_dep); flush(&cnt->n_secondary, c_sec);
}

// ------------------------------------------------------------------ K5: batch statistics (Reading R8)
// One voxel per thread (L140): dose of each batch (Gy per primary) from its tally, running mean and sum of squared
// deviations over the B batches (Welford), then mean dose and standard error.
__global__ void __launch_bounds__(256) stats_kernel(Tables T, Grid G, const float *tally, float *dose, float *sigma, int B,
                                                    uint64_t n_total, uint32_t nvox) {
  // four consecutive voxels per thread (16-byte loads from each batch grid keep enough bytes in flight for HBM);
  // a ragged tail or an unaligned grid size falls back to one voxel per thread
  const bool vec = (nvox & 3u) == 0u;
  const uint32_t nitems = vec ? nvox >> 2 : nvox;
  const float ib = 1.0f / ((float)B * (float)(B - 1));
  for (uint32_t it = blockIdx.x * blockDim.x + threadIdx.x; it < nitems; it += gridDim.x * blockDim.x) {
    const uint32_t v0 = vec ? it << 2 : it; const int nv = vec ? 4 : 1;
    float inv_m[4], mu[4] = {0.f, 0.f, 0.f, 0.f}, s[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      if (k < nv) {
        const int hu = G.hu[v0 + k];
        const MatBin &m = T.bins[hu_to_bin(T, T.hu_lut, hu)];
        inv_m[k] = 1.602176634e-10f / (bin_density(m, hu) * G.vol);
      } else inv_m[k] = 0.f;
    }
    for (int b = 0; b < B; ++b) {
      const uint64_t h0 = ((uint64_t)b * n_total + B - 1) / B, h1 = ((uint64_t)(b + 1) * n_total + B - 1) / B;
      const float inb = h1 > h0 ? 1.0f / (float)(h1 - h0) : 0.f, ibp = 1.0f / (float)(b + 1);
      float t[4] = {0.f, 0.f, 0.f, 0.f};
      if (vec) { const float4 q = *reinterpret_cast<const float4 *>(tally + (size_t)b * nvox + v0); t[0] = q.x; t[1] = q.y; t[2] = q.z; t[3] = q.w; }
      else t[0] = tally[(size_t)b * nvox + v0];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const float d = t[k] * inv_m[k] * inb;
        const float delta = d - mu[k]; mu[k] += delta * ibp; s[k] += delta * (d - mu[k]);
      }
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      if (k < nv) {
        dose[v0 + k] = mu[k];
        const float var = s[k] * ib;
        sigma[v0 + k] = var > 0.f ? sqrtf(var) : 0.f;
      }
    }
  }
}

// influence matrix MeV -> Gy per primary history of the call: D[i][j] *= Gy/(MeV/g) / (rho_j V n)
__global__ void __launch_bounds__(256) influence_finish_kernel(Tables T, Grid G, const int32_t *roi_vox, uint32_t n_roi, uint32_t nspots,
                                                               float inv_n, float *dij) {
  const size_t total = (size_t)n_roi * nspots;
  for (size_t k = blockIdx.x * (size_t)blockDim.x + threadIdx.x; k < total; k += (size_t)gridDim.x * blockDim.x) {
    const int hu = G.hu[roi_vox[k % n_roi]];
    const MatBin &m = T.bins[hu_to_bin(T, T.hu_lut, hu)];
    dij[k] *= 1.602176634e-10f * inv_n / (bin_density(m, hu) * G.vol);
  }
}

// LET_d = sum(e x LET) / sum(e) per voxel (keV/um), 0 where no proton step deposited energy
__global__ void __launch_bounds__(256) letd_kernel(const float *num, const float *den, float *out, uint32_t nvox) {
  for (uint32_t v = blockIdx.x * blockDim.x + threadIdx.x; v < nvox; v += gridDim.x * blockDim.x)
    out[v] = den[v] > 0.f ? num[v] / den[v] : 0.f;
}

}  // namespace pmc
