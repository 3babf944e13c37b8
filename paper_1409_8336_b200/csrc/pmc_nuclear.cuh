// pmc_nuclear.cuh — non-elastic proton-nucleus collisions: Bertini-style intranuclear cascade (
// Reading R6) followed by evaporation (Reading R7), as device functions plus the event-queue
// kernels of the transport scheduler and the standalone kernel behind pmc_nonelastic.
//
// Precision: cascade geometry, sampling and NN kinematics run in fp32; the conservation bookkeeping (sums of
// outgoing four-momenta, residual excitation energy, two-body decay of the compound nucleus, separation
// energies) runs in fp64 because it subtracts nuclear masses of 1e4 MeV to get MeV-scale answers.  Charge and
// baryon number are integers throughout.
#pragma once
#include "pmc_device.cuh"
#include "pmc_transport.cuh"

namespace pmc {

// Fixed capacities of a cascade attempt; an attempt that needs more is abandoned and repeated like one that trips the step
// guard, and counted (pmc_counters.n_inc_cap_trips).  The oracle (limit 200 / none) never saw more than 7 waiting and 7
// outgoing nucleons in 1e6 events each of p + 48Ti at 230 MeV, p + 16O at 200 MeV and p + 40Ca at 70 MeV.
constexpr int CASC_STACK = 16;      // cascade nucleons waiting to be tracked
constexpr int MAX_INC_OUT = 16;     // nucleons leaving the nucleus in one cascade
constexpr int MAX_SEC = 48;         // records per event in the standalone kernel's slot buffer (INC + evaporation + residual)
constexpr int MAX_INC_STEPS = 1024; // tracking steps per attempt before it is abandoned and repeated (Reading R6.8)
constexpr int NQ = 64;              // quadrature bins of the evaporation spectrum (Reading R7)

struct SecRec { int16_t Z, A; uint8_t origin, pad[3]; float ke; float dir[3]; };   // == pmc_secondary (24 B)
static_assert(sizeof(SecRec) == 24, "pmc_secondary layout");

struct OutNuc { int type; float ke; V3 dir; };                                   // type 0 proton, 1 neutron
struct Residual { int Z, A; double estar; double P[3]; double mass_gs; };
struct CascNucleon { V3 r, p; int type, shell; };

__device__ __forceinline__ float nucleon_mass(int type) { return type == 0 ? MP : MN; }
__device__ __forceinline__ double nmass(const Tables &T, int z, int a) {
  return (z < 0 || a < 1 || z >= T.zdim || a >= T.adim || z > a) ? 0.0 : T.mass[z * T.adim + a];
}

// Per-lane state of one cascade attempt.  The cascade is written as a state machine (begin / step / finalize) so
// that the 32 lanes of a warp execute the same step of 32 different cascades together: a thread-per-event loop nest
// with early exits leaves the lanes serialised (measured: 1.4 active lanes per instruction).
struct IncLane {
  CascNucleon stack[CASC_STACK]; OutNuc out[MAX_INC_OUT];
  CascNucleon c;
  int sp, ncoll, n_out, np_out, guard; bool alive, failed;
  int trip;                       // why the attempt was abandoned: 1 step guard, 2 stack full, 4 out-list full
  int hw_stack, hw_out;           // high-water marks over the lane's attempts
  double e_out_sum, pxs, pys, pzs;
};

// entry: uniform over the disc of radius rmax, travelling along +z (L75 "random point of entry"); refraction into
// the outermost shell: gains V, tangential momentum conserved
__device__ __forceinline__ void inc_begin(const Nucleus &N, float t_in, RngK &g, const RoundKeys &K, IncLane &L) {
  const int ns = N.nshell;
  L.sp = 0; L.ncoll = 0; L.n_out = 0; L.np_out = 0; L.guard = 0; L.failed = false; L.trip = 0;
  L.e_out_sum = 0; L.pxs = 0; L.pys = 0; L.pzs = 0;
  const uint4 r = g.next4(K);
  const float b = N.rmax * sqrtf(u01(r.x)); float sph, cph; sincospif(2.0f * u01(r.y), &sph, &cph);
  const V3 r0{b * cph, b * sph, -sqrtf(fmaxf(0.f, N.rmax * N.rmax - b * b))};
  const float Tn = t_in + N.V[0][ns - 1], p0 = sqrtf(t_in * (t_in + 2.0f * MP)), p1 = sqrtf(Tn * (Tn + 2.0f * MP));
  const V3 nh = unit(r0), pv{0.f, 0.f, p0};
  const float pr = dot(pv, nh); const V3 pt = pv - pr * nh;
  const float pr2 = p1 * p1 - dot(pt, pt);
  L.c = {r0, pt + (-sqrtf(fmaxf(pr2, 0.f))) * nh, 0, ns - 1};
  L.alive = true;
}
__device__ __forceinline__ void inc_fail(IncLane &L) { L.failed = true; L.alive = false; L.sp = 0; }

// direction uniform on the sphere from two 16-bit fields
__device__ __forceinline__ V3 isotropic16(uint32_t a16, uint32_t b16) {
  const float c = fmaf(2.0f, u16f(a16), -1.0f), s = fsqrt(fmaxf(0.f, fmaf(-c, c, 1.0f)));
  float sp, cp; sincos_2pi(u16f(b16), &sp, &cp);
  return {s * cp, s * sp, c};
}
// one step of the nucleon being tracked: candidate collisions vs shell boundary (Reading R6.3-R6.5)
__device__ __forceinline__ void inc_step(const Nucleus &N, RngK &g, const RoundKeys &K, IncLane &L) {
  CascNucleon &c = L.c;
  const int ns = N.nshell;
  if (++L.guard > MAX_INC_STEPS) { L.trip = 1; inc_fail(L); return; }   // bound orbit in a dilute shell (Reading R6.8)
  const int k = c.shell, ty = c.type;
  const float m = nucleon_mass(ty), p2 = dot(c.p, c.p), E = fsqrt(p2 + m * m), Tk = fdiv(p2, E + m);
  const V3 d = frsq(p2) * c.p;
  // candidate collisions with a nucleon of the projectile's own type and with one of the other type, both from the Fermi
  // sea (Reading R6.3).  One Philox block serves both: per partner 16 bits each for |q|^3, cos, azimuth and free path.
  // Looping over same / other (instead of proton / neutron) keeps the lanes of a warp on the same cross-section formula.
  float dbest = BIG, plab_best = 0.f; int tbest = -1; V3 qbest{0.f, 0.f, 0.f};
  const uint4 rq = g.next4(K);
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    const int tp = s == 0 ? ty : 1 - ty;
    const float rho = N.rho[tp][k];
    if (rho <= 0.f) continue;
    const uint32_t wa = s == 0 ? rq.x : rq.z, wb = s == 0 ? rq.y : rq.w;
    const float mq = nucleon_mass(tp), qmag = N.pF[tp][k] * fex2(flg2(u16f(wa >> 16)) * (1.0f / 3.0f));
    const V3 q = qmag * isotropic16(wa & 0xFFFFu, wb >> 16);
    const float Eq = fsqrt(fmaf(qmag, qmag, mq * mq));
    const float e1 = (E * Eq - dot(c.p, q)) * (tp == 0 ? 1.0f / MP : 1.0f / MN);                       // projectile energy in the partner rest frame
    const float plab = fsqrt(fmaxf(fmaf(e1, e1, -m * m), 0.f));
    const float sig = N.const_sigma_mb >= 0.f ? N.const_sigma_mb : (s == 0 ? cug_sigma_pp(plab * 1e-3f) : cug_sigma_np(plab * 1e-3f));
    const float dist = -LN2 * flg2(u16f(wb & 0xFFFFu)) * frcp(rho * sig * 0.1f);  // 1 mb = 0.1 fm^2
    if (dist < dbest) { dbest = dist; tbest = tp; qbest = q; plab_best = plab; }
  }
  // distance to the shell boundaries along d
  const float rr = dot(c.r, c.r), bq = dot(c.r, d), r_out = N.rout[k], r_in = k > 0 ? N.rout[k - 1] : 0.f;
  float dbound = -bq + fsqrt(fmaxf(bq * bq - (rr - r_out * r_out), 0.f)); bool inward = false;
  if (k > 0 && bq < 0.f) {
    const float disc = bq * bq - (rr - r_in * r_in);
    if (disc > 0.f) { const float s_in = -bq - fsqrt(disc); if (s_in < dbound) { dbound = fmaxf(s_in, 0.f); inward = true; } }
  }
  if (dbest < dbound) {
    // ---- collision attempt (Reading R6.4)
    c.r = c.r + dbest * d;
    const int tp = tbest; const float mq = nucleon_mass(tp);
    const V3 q = qbest; const float Eq = fsqrt(dot(q, q) + mq * mq);
    const V3 Pt = c.p + q; const float Et = E + Eq; const V3 beta = fdiv(1.0f, Et) * Pt;
    const float s = Et * Et - dot(Pt, Pt);
    const float pcm = fsqrt(fmaxf((s - (m + mq) * (m + mq)) * (s - (m - mq) * (m - mq)), 0.f) * fdiv(0.25f, s));
    V3 p1 = c.p; float E1 = E; boost(-1.0f * beta, p1, E1);             // projectile in the CM
    const V3 ax = unit(p1);
    const uint4 r = g.next4(K);
    const float ct = sample_nn_cos(tp == ty, plab_best * 1e-3f, pcm, r.x, r.y), st = fsqrt(fmaxf(0.f, 1.0f - ct * ct));
    float sph, cph; sincos_2pi(u01(r.z), &sph, &cph);
    V3 n1 = pcm * to_lab(ax, st * cph, st * sph, ct), n2 = -1.0f * n1;
    float En1 = fsqrt(pcm * pcm + m * m), En2 = fsqrt(pcm * pcm + mq * mq);
    boost(beta, n1, En1); boost(beta, n2, En2);
    const float T1 = En1 - m, T2 = En2 - mq;
    const bool ok = !N.pauli || (T1 > N.EF[ty][k] && T2 > N.EF[tp][k]);  // L77 Pauli blocking
    if (!ok) return;                                                     // blocked: go on unchanged
    L.ncoll++;
    // trapping (Reading R6.4): outside energy eps = T - V <= B_C stays in the nucleus
    const float bc2 = tp == 0 ? N.coulomb : 0.f, bc1 = ty == 0 ? N.coulomb : 0.f;
    if (T2 - N.V[tp][k] > bc2) {
      if (L.sp >= CASC_STACK) { L.trip = 2; inc_fail(L); return; }
      L.stack[L.sp++] = {c.r, n2, tp, k};
      L.hw_stack = max(L.hw_stack, L.sp);
    }
    if (T1 - N.V[ty][k] > bc1) c.p = n1; else L.alive = false;
    return;
  }
  // ---- shell boundary (L77 "reflection and refraction"; Reading R6.5)
  c.r = c.r + dbound * d;
  const float rb = inward ? r_in : r_out;
  c.r = (rb * frsq(dot(c.r, c.r))) * c.r;
  const V3 nh = fdiv(1.0f, rb) * c.r;
  const float pr = dot(c.p, nh); const V3 pt = c.p - pr * nh;
  const int k2 = inward ? k - 1 : k + 1;
  const float Vnew = k2 >= ns ? 0.f : N.V[ty][k2], T2 = Tk + (Vnew - N.V[ty][k]);
  const float pn2 = T2 > 0.f ? T2 * (T2 + 2.0f * m) : -1.0f, pr2 = pn2 - dot(pt, pt);
  if (pn2 <= 0.f || pr2 <= 0.f) { c.p = pt - pr * nh; return; }           // specular reflection
  const V3 pnew = pt + ((pr > 0.f ? 1.0f : -1.0f) * fsqrt(pr2)) * nh;
  if (k2 >= ns) {                                                       // leaves the nucleus with KE = eps
    if (L.n_out >= MAX_INC_OUT) { L.trip = 4; inc_fail(L); return; }
    OutNuc &o = L.out[L.n_out++];
    L.hw_out = max(L.hw_out, L.n_out);
    o.type = ty; o.ke = T2; o.dir = unit(pnew);
    L.e_out_sum += (double)T2 + (ty == 0 ? MP_D : MN_D); L.pxs += pnew.x; L.pys += pnew.y; L.pzs += pnew.z;
    if (ty == 0) L.np_out++;
    L.alive = false;
  } else { c.p = pnew; c.shell = k2; }
}

// end of an attempt: false if no Pauli-allowed collision happened or the outcome is invalid (L75); else the
// residual nucleus (Reading R6.7): exact integers, relativistic invariant mass, fp64
__device__ __forceinline__ bool inc_finalize(const Tables &T, const Nucleus &N, float t_in, const IncLane &L, Residual &res) {
  if (L.failed || L.ncoll == 0) return false;                               // L75: need >= 1 allowed collision
  const int Ar = N.A + 1 - L.n_out, Zr = N.Z + 1 - L.np_out;
  const double Mgs = nmass(T, Zr, Ar);
  if (Ar < 1 || Zr < 0 || Zr > Ar || Mgs <= 0) return false;
  const double tin = (double)t_in, pin = sqrt(tin * (tin + 2 * MP_D));
  const double Eres = (tin + MP_D + N.mass) - L.e_out_sum, Px = -L.pxs, Py = -L.pys, Pz = pin - L.pzs;
  const double M2 = Eres * Eres - (Px * Px + Py * Py + Pz * Pz);
  if (Eres <= 0 || M2 <= 0) return false;
  const double estar = sqrt(M2) - Mgs;
  if (estar < 0) return false;
  if (Ar == 1 && estar > 1e-4) return false;                                // a lone nucleon cannot be excited
  res.Z = Zr; res.A = Ar; res.estar = estar; res.P[0] = Px; res.P[1] = Py; res.P[2] = Pz; res.mass_gs = Mgs;
  return true;
}
// Reading R6.8 (never reached in the configs): after 1e5 failed attempts form the compound nucleus (Z+1, A+1)
__device__ __forceinline__ void inc_compound(const Tables &T, const Nucleus &N, float t_in, Residual &res) {
  const double tin = (double)t_in, pin = sqrt(tin * (tin + 2 * MP_D)), Et = tin + MP_D + N.mass, Mgs = nmass(T, N.Z + 1, N.A + 1);
  res.Z = N.Z + 1; res.A = N.A + 1; res.estar = sqrt(Et * Et - pin * pin) - Mgs; res.P[0] = 0; res.P[1] = 0; res.P[2] = pin; res.mass_gs = Mgs;
}

// Warp-synchronous cascade engine: every lane owns one event at a time and all 32 lanes take one cascade step per
// trip of the loop; a lane whose event is done fetches the next one from the shared counter `head` (warp-aggregated).
// load(i, N, t_in, g) sets up event i; store(i, g, out, n_out, R) consumes its result.  L75: the attempt is repeated
// (fresh draws of the same stream) until it has at least one Pauli-allowed collision and a valid residual.
// All 32 lanes of every warp must call.
struct IncStats { unsigned long long tries = 0, guard = 0, cap = 0; int hw_stack = 0, hw_out = 0; };
template <class Load, class Store>
__device__ __forceinline__ void inc_machine(const Tables &T, const RoundKeys &K, uint32_t n, uint32_t *head, IncStats &st,
                                            Load load, Store store) {
  // Lane states.  STEP: tracking a nucleon.  WAIT: attempt finished (needs finalize, then store + next event, or a
  // fresh attempt) or no event yet.  DONE: queue exhausted.  The turnover work of WAIT lanes is divergent and long
  // compared with one step, so it is batched: it runs when TURNOVER lanes are waiting (or nobody can step), not
  // every time a single lane finishes.
  enum { STEP = 0, WAIT = 1, DONE = 2 };
  constexpr int TURNOVER = 8;
  IncLane L; L.alive = false; L.sp = 0; L.failed = false; L.trip = 0; L.hw_stack = 0; L.hw_out = 0;
  const Nucleus *N = nullptr; float t_in = 0.f; RngK g; uint32_t ev = 0; int ntry = 0;
  bool busy = false; int state = WAIT;
  const int lane = threadIdx.x & 31;
  while (true) {
    const unsigned waiting = __ballot_sync(0xffffffffu, state == WAIT), stepping = __ballot_sync(0xffffffffu, state == STEP);
    if (!waiting && !stepping) break;
    if (waiting && (__popc(waiting) >= TURNOVER || !stepping)) {
      if (state == WAIT && busy) {                       // end of an attempt
        if (L.trip == 1) st.guard++; else if (L.trip) st.cap++;
        Residual R;
        if (inc_finalize(T, *N, t_in, L, R)) { store(ev, g, L.out, L.n_out, R); busy = false; }
        else if (ntry >= 100000) { inc_compound(T, *N, t_in, R); store(ev, g, L.out, 0, R); busy = false; }
        else { ++ntry; st.tries++; inc_begin(*N, t_in, g, K, L); state = STEP; }
      }
      __syncwarp();
      const unsigned need = __ballot_sync(0xffffffffu, state == WAIT && !busy);
      if (need) {                                        // next events, warp-aggregated fetch
        const int leader = __ffs(need) - 1;
        uint32_t base = 0;
        if (lane == leader) base = atomicAdd(head, (uint32_t)__popc(need));
        base = __shfl_sync(0xffffffffu, base, leader);
        if (state == WAIT && !busy) {
          ev = base + (uint32_t)__popc(need & ((1u << lane) - 1u));
          if (ev < n) { load(ev, N, t_in, g); busy = true; ntry = 1; st.tries++; inc_begin(*N, t_in, g, K, L); state = STEP; }
          else state = DONE;
        }
      }
      __syncwarp();
    }
    if (state == STEP) {
      inc_step(*N, g, K, L);
      if (!L.alive) {
        if (L.sp > 0) { L.c = L.stack[--L.sp]; L.alive = true; }
        else state = WAIT;
      }
    }
    __syncwarp();
  }
  st.hw_stack = L.hw_stack; st.hw_out = L.hw_out;
}
// all 32 lanes must call
__device__ __forceinline__ void flush_inc_stats(Counters *cnt, const IncStats &st) {
  flush(&cnt->n_inc_tries, st.tries); flush(&cnt->n_inc_guard, st.guard); flush(&cnt->n_inc_cap, st.cap);
  const int hs = __reduce_max_sync(0xffffffffu, st.hw_stack), ho = __reduce_max_sync(0xffffffffu, st.hw_out);
  if ((threadIdx.x & 31) == 0) { atomicMax(&cnt->inc_max_stack, (unsigned)hs); atomicMax(&cnt->inc_max_out, (unsigned)ho); }
}

// ------------------------------------------------------------------ evaporation (Reading R7)
__constant__ int EJ_Z[6] = {0, 1, 1, 1, 2, 2};
__constant__ int EJ_A[6] = {1, 1, 2, 3, 3, 4};
__constant__ float EJ_SPIN_G[6] = {2.f, 2.f, 3.f, 2.f, 2.f, 1.f};
__device__ __forceinline__ float pairing(int Z, int A) {
  const int N = A - Z; const float d = 12.0f * rsqrtf((float)A);
  return (Z % 2 == 0 && N % 2 == 0) ? 2.0f * d : ((Z % 2) != (N % 2) ? d : 0.f);
}
// One open channel.  The integrand of its width, P_j(e) = pref sigma_inv(e) e exp(2 sqrt(a_d (emax - e)) - ref), is kept in
// the form (s1 e + s0) 2^(A sqrt(emax - e) - B): sigma_inv(e) e is linear in e for Dostrovsky's inverse cross-sections
// (alpha (e + beta) for neutrons, (1 + c_j)(e - k_j V_j) for charged ejectiles), so a quadrature point costs two MUFU
// and five FMA-class instructions.
struct Chan { float S, emin, emax, s1, s0, A, B; int Zd, Ad; double Md, mj; };
__device__ bool chan_setup(const Tables &T, int Z, int A, float estar, double Mpar, int j, float ref, Chan &c) {
  const int Zd = Z - EJ_Z[j], Ad = A - EJ_A[j];
  if (Ad < 2 || Zd < 0) return false;
  const double Md = nmass(T, Zd, Ad), mj = nmass(T, EJ_Z[j], EJ_A[j]);
  if (Md <= 0) return false;
  c.Zd = Zd; c.Ad = Ad; c.Md = Md; c.mj = mj; c.S = (float)(Md + mj - Mpar);
  const float a13 = cbrtf((float)Ad);
  float kV = 0.f, cj = 0.f;
  if (j > 0) {
    const float rhoj = j == 1 ? 0.f : 1.2f, V = 1.44f * EJ_Z[j] * Zd / (1.5f * a13 + rhoj);
    kV = T.evap_k[j * T.zdim + Zd] * V; cj = T.evap_c[j * T.zdim + Zd];
  }
  c.emin = kV; c.emax = estar - c.S - pairing(Zd, Ad);
  if (c.emax <= c.emin) return false;
  const float alpha = 0.76f + 2.2f / a13, beta = (2.12f / (a13 * a13) - 0.050f) / alpha;
  const float pref = EJ_SPIN_G[j] * (float)mj * a13 * a13;
  c.s1 = pref * (j == 0 ? alpha : 1.0f + cj); c.s0 = j == 0 ? c.s1 * beta : -c.s1 * kV;
  c.A = 2.0f * LOG2E * sqrtf(Ad * 0.125f); c.B = ref * LOG2E;
  return true;
}
// Midpoint i of the NQ bins of [emin, emax]: e_i = emin + (i + 1/2) de, emax - e_i = (NQ - 1/2 - i) de, so that
// P(e_i) = (lin1 (i + 1/2) + lin0) 2^(Ade sqrt(NQ - 1/2 - i) - B) with the square roots a constant table (filled by
// pmc_create): one MUFU and three FMAs per point.
__constant__ float EVAP_SQ[NQ];
struct ChanQ { float lin0, lin1, Ade, B; };
__device__ __forceinline__ ChanQ chan_quad(const Chan &c, float de) { return {fmaf(c.s1, c.emin, c.s0), c.s1 * de, c.A * fsqrt(de), c.B}; }
__device__ __forceinline__ float chan_f(const ChanQ &q, int i) {
  return fmaf(q.lin1, (float)i + 0.5f, q.lin0) * fex2(fmaf(q.Ade, EVAP_SQ[i], -q.B));
}
struct Emission { int j; float ke; V3 dir; };
// one emission from R (updated in place); returns false when no channel is open
__device__ bool evap_emit(const Tables &T, Residual &R, Rng &g, uint32_t mask, Emission &em, float *eps_out, float *cos_out) {
  const float estar = (float)R.estar;
  const float ref = 2.0f * sqrtf(R.A * 0.125f * fmaxf(estar, 0.f));
  float width[6]; float tot = 0.f;
#pragma unroll 1
  for (int j = 0; j < 6; ++j) {
    width[j] = 0.f;
    Chan c;
    if (!((mask >> j) & 1u) || !chan_setup(T, R.Z, R.A, estar, R.mass_gs, j, ref, c)) continue;
    const float de = (c.emax - c.emin) * (1.0f / NQ);
    const ChanQ q = chan_quad(c, de);
    float w = 0.f;
#pragma unroll
    for (int i = 0; i < NQ; ++i) w += chan_f(q, i);
    width[j] = w * de; tot += width[j];
  }
  if (!(tot > 0.f)) return false;
  const uint4 r = g.next4();
  float u = u01(r.x) * tot; int j = -1;
#pragma unroll
  for (int q = 0; q < 6; ++q) if (width[q] > 0.f && (j < 0 || u >= 0.f)) { j = q; u -= width[q]; }
  Chan c; chan_setup(T, R.Z, R.A, estar, R.mass_gs, j, ref, c);
  const float de = (c.emax - c.emin) * (1.0f / NQ);
  float v = u01(r.y) * width[j] / de; int bin = NQ - 1;
  const ChanQ cq = chan_quad(c, de);
  for (int i = 0; i < NQ; ++i) { const float f = chan_f(cq, i); if (v < f) { bin = i; break; } v -= f; }
  const float eps = c.emin + ((float)bin + u01(r.z)) * de;                  // total CM kinetic energy released
  // relativistic two-body decay of M* -> m_j + M_d* (isotropic in the nucleus rest frame, L79), fp64
  const uint4 r2 = g.next4();
  const V3 dirc = isotropic(r2.x, r2.y);
  const double mj = c.mj, Mstar = R.mass_gs + R.estar, Ud = R.estar - (c.Md + mj - R.mass_gs) - (double)eps, Md = c.Md + Ud;
  const double pc2 = (Mstar * Mstar - (mj + Md) * (mj + Md)) * (Mstar * Mstar - (mj - Md) * (mj - Md)) / (4 * Mstar * Mstar);
  const double pc = sqrt(fmax(pc2, 0.0));
  double pj[3] = {pc * dirc.x, pc * dirc.y, pc * dirc.z};
  double Ej = sqrt(pc * pc + mj * mj), Ed = sqrt(pc * pc + Md * Md);
  const double Epar = sqrt(R.P[0] * R.P[0] + R.P[1] * R.P[1] + R.P[2] * R.P[2] + Mstar * Mstar);
  const double bx = R.P[0] / Epar, by = R.P[1] / Epar, bz = R.P[2] / Epar, b2 = bx * bx + by * by + bz * bz;
  double pd[3] = {-pj[0], -pj[1], -pj[2]};
  if (b2 > 0) {
    const double gam = 1.0 / sqrt(1.0 - b2);
    const double bpj = bx * pj[0] + by * pj[1] + bz * pj[2], fj = (gam - 1.0) * bpj / b2 + gam * Ej;
    pj[0] += fj * bx; pj[1] += fj * by; pj[2] += fj * bz; Ej = gam * (Ej + bpj);
    const double bpd = -bpj + 0.0, fd = (gam - 1.0) * bpd / b2 + gam * Ed;
    pd[0] += fd * bx; pd[1] += fd * by; pd[2] += fd * bz; Ed = gam * (Ed + bpd);
  }
  const double pn = sqrt(pj[0] * pj[0] + pj[1] * pj[1] + pj[2] * pj[2]);
  em.j = j; em.ke = (float)(Ej - mj);
  em.dir = pn > 0 ? V3{(float)(pj[0] / pn), (float)(pj[1] / pn), (float)(pj[2] / pn)} : V3{0.f, 0.f, 1.f};
  R.Z = c.Zd; R.A = c.Ad; R.estar = Ud; R.P[0] = pd[0]; R.P[1] = pd[1]; R.P[2] = pd[2]; R.mass_gs = c.Md;
  if (eps_out) *eps_out = eps;
  if (cos_out) *cos_out = dirc.z;
  return true;
}
__device__ __forceinline__ double residual_ke(const Residual &R) {
  const double Mres = R.mass_gs + R.estar, p2 = R.P[0] * R.P[0] + R.P[1] * R.P[1] + R.P[2] * R.P[2];
  return p2 / (sqrt(p2 + Mres * Mres) + Mres);
}

// Warp-synchronous evaporation engine (same scheme as inc_machine): one emission per lane per trip of the loop.
// load(i, R, g) sets up residual i; emit(i, g, em) consumes one emitted particle; done(i, g, R) the final residual.
template <class Load, class Emit, class Done>
__device__ __forceinline__ void evap_machine(const Tables &T, uint32_t n, uint32_t *head, Load load, Emit emit, Done done) {
  Residual R; Rng g; uint32_t ev = 0; int nem = 0;
  bool busy = false, exhausted = false;
  const int lane = threadIdx.x & 31;
  while (true) {
    const unsigned need = __ballot_sync(0xffffffffu, !busy && !exhausted);
    if (need) {
      const int leader = __ffs(need) - 1;
      uint32_t base = 0;
      if (lane == leader) base = atomicAdd(head, (uint32_t)__popc(need));
      base = __shfl_sync(0xffffffffu, base, leader);
      if (!busy && !exhausted) {
        ev = base + (uint32_t)__popc(need & ((1u << lane) - 1u));
        if (ev < n) { load(ev, R, g); busy = true; nem = 0; }
        else exhausted = true;
      }
    }
    if (!__any_sync(0xffffffffu, busy)) break;
    Emission em; bool ok = false;
    if (busy) ok = nem < 200 && evap_emit(T, R, g, 0x3Fu, em, nullptr, nullptr);
    __syncwarp();
    if (busy) {
      if (ok) { ++nem; emit(ev, g, em); }
      else { done(ev, g, R); busy = false; }
    }
  }
}

// ------------------------------------------------------------------ event-queue kernels of the transport scheduler
struct ResQueue { Queue q; uint32_t *za; float *px, *py, *pz; };   // q.e = E*, q.aux = spot << 8 | next product index

// K3: intranuclear cascades over the non-elastic queue (PAPER.md:L128(3), L136), one event per lane at a time
__global__ void __launch_bounds__(128) inc_kernel(Tables T, RunParams P, Queue in, uint32_t *head, Queue out, ResQueue rq,
                                                  float *tally, Counters *cnt) {
  const uint32_t n = min(*in.count, in.cap);
  double c_dep = 0, c_neu = 0, c_q = 0; unsigned long long c_sec = 0; IncStats st;
  Particle p;
  auto load = [&](uint32_t i, const Nucleus *&N, float &t_in, RngK &g) {
    p = queue_load(in, i);
    g.init(P.hist0 + p.hist, p.pid, p.blk);
    N = &T.nuc[aux_low(p.aux)]; t_in = p.e;
  };
  auto store = [&](uint32_t, RngK &g, const OutNuc *outn, int n_out, const Residual &R) {
    const Nucleus &N = T.nuc[aux_low(p.aux)];
    float dep = 0.f; uint32_t kchild = 0; double msum = 0;
    for (int k = 0; k < n_out; ++k) {
      const OutNuc &o = outn[k];
      msum += o.type == 0 ? MP_D : MN_D;
      if (o.type == 0) {                                                   // L79: only protons are followed
        if (o.ke > T.e_cut) {
          Particle s = p; s.d = unit(to_lab(p.d, o.dir.x, o.dir.y, o.dir.z)); s.e = o.ke;
          s.pid = g.child_id(P.rk, kchild++); s.blk = 0u; s.aux = aux_with(p.aux, 0u); c_sec++;
          if (!queue_push(out, s)) atomicOr(&cnt->overflow, 16u);
        } else dep += o.ke;
      } else c_neu += (double)o.ke;                                        // neutrons: not transported
    }
    c_q += msum + R.mass_gs - MP_D - N.mass;
    if (dep != 0.f) { atomicAdd(tally + batch_base(P, p.hist) + (uint32_t)p.vox, dep); c_dep += (double)dep; score_influence(P, p.aux, p.vox, dep); }
    // residual -> evaporation queue (keeps the event frame: p.d is the incident direction)
    const uint32_t slot = warp_alloc(rq.q.count);
    if (slot >= rq.q.cap) atomicOr(&cnt->overflow, 32u);
    else {
      const Queue &q = rq.q;
      q.x[slot] = p.r.x; q.y[slot] = p.r.y; q.z[slot] = p.r.z; q.u[slot] = p.d.x; q.v[slot] = p.d.y; q.w[slot] = p.d.z;
      q.e[slot] = (float)R.estar; q.vox[slot] = p.vox; q.hist[slot] = p.hist; q.pid[slot] = p.pid; q.blk[slot] = g.blk;
      q.aux[slot] = aux_with(p.aux, kchild); rq.za[slot] = ((uint32_t)R.Z << 16) | (uint32_t)R.A;
      rq.px[slot] = (float)R.P[0]; rq.py[slot] = (float)R.P[1]; rq.pz[slot] = (float)R.P[2];
    }
  };
  inc_machine(T, P.rk, n, head, st, load, store);
  flush(&cnt->e_deposit, c_dep); flush(&cnt->e_neutron, c_neu); flush(&cnt->e_q, c_q);
  flush(&cnt->n_secondary, c_sec); flush_inc_stats(cnt, st);
}

// K4: nuclear de-excitations over the residual queue (PAPER.md:L128(4), L136), one residual per lane at a time
__global__ void __launch_bounds__(128) evap_kernel(Tables T, RunParams P, ResQueue rq, uint32_t *head, Queue out, float *tally,
                                                   Counters *cnt) {
  const uint32_t n = min(*rq.q.count, rq.q.cap);
  double c_dep = 0, c_neu = 0, c_q = 0, c_gam = 0; unsigned long long c_sec = 0;
  Particle p; double m0 = 0, msum = 0; uint32_t kchild = 0; float dep = 0.f;
  auto load = [&](uint32_t i, Residual &R, Rng &g) {
    p = queue_load(rq.q, i);
    g.init(P.seed, P.hist0 + p.hist, p.pid, p.blk);
    R.Z = (int)(rq.za[i] >> 16); R.A = (int)(rq.za[i] & 0xffffu); R.estar = (double)p.e;
    R.P[0] = rq.px[i]; R.P[1] = rq.py[i]; R.P[2] = rq.pz[i]; R.mass_gs = nmass(T, R.Z, R.A);
    m0 = R.mass_gs; msum = 0; kchild = aux_low(p.aux); dep = 0.f;
  };
  auto emit = [&](uint32_t, Rng &g, const Emission &em) {
    msum += nmass(T, EJ_Z[em.j], EJ_A[em.j]);
    if (em.j == 1) {
      if (em.ke > T.e_cut) {
        Particle s = p; s.d = unit(to_lab(p.d, em.dir.x, em.dir.y, em.dir.z)); s.e = em.ke;
        s.pid = g.child_id(kchild++); s.blk = 0u; s.aux = aux_with(p.aux, 0u); c_sec++;
        if (!queue_push(out, s)) atomicOr(&cnt->overflow, 64u);
      } else dep += em.ke;
    } else if (em.j == 0) c_neu += (double)em.ke;
    else dep += em.ke;                                                     // d, t, 3He, alpha: local (L79)
  };
  auto done = [&](uint32_t, Rng &, const Residual &R) {
    const double kres = residual_ke(R);
    if (R.A == 1 && R.Z == 0) c_neu += kres; else dep += (float)kres;
    c_gam += R.estar;                                                       // L79: no photon evaporation
    c_q += msum + R.mass_gs - m0;
    if (dep != 0.f) { atomicAdd(tally + batch_base(P, p.hist) + (uint32_t)p.vox, dep); c_dep += (double)dep; score_influence(P, p.aux, p.vox, dep); }
  };
  evap_machine(T, n, head, load, emit, done);
  flush(&cnt->e_deposit, c_dep); flush(&cnt->e_neutron, c_neu); flush(&cnt->e_q, c_q); flush(&cnt->e_gamma, c_gam);
  flush(&cnt->n_secondary, c_sec);
}

// ------------------------------------------------------------------ standalone non-elastic events (pmc_nonelastic; Table I)
// Two kernels like the scheduler's (cascade, then de-excitation); event i of the call uses the stream (seed, ev0 + i).
struct ResRec { int Z, A; double estar; double P[3]; uint32_t blk; int zs, as; };

__global__ void __launch_bounds__(128) nonelastic_inc_kernel(Tables T, const Nucleus *nuc, float t_in0, RoundKeys K, uint64_t ev0,
                                                             uint32_t n, uint32_t *head, SecRec *slots, uint32_t *counts,
                                                             ResRec *res, Counters *cnt) {
  IncStats st;
  auto load = [&](uint32_t i, const Nucleus *&N, float &t_in, RngK &g) { g.init(ev0 + i, 0u, 0u); N = nuc; t_in = t_in0; };
  auto store = [&](uint32_t i, RngK &g, const OutNuc *outn, int n_out, const Residual &R) {
    SecRec *s = slots + (size_t)i * MAX_SEC; int zs = 0;
    for (int k = 0; k < n_out; ++k) {
      SecRec rec{}; rec.Z = outn[k].type == 0 ? 1 : 0; rec.A = 1; rec.origin = 0; rec.ke = outn[k].ke;
      rec.dir[0] = outn[k].dir.x; rec.dir[1] = outn[k].dir.y; rec.dir[2] = outn[k].dir.z;
      zs += rec.Z; s[k] = rec;
    }
    counts[i] = (uint32_t)n_out;
    ResRec rr; rr.Z = R.Z; rr.A = R.A; rr.estar = R.estar; rr.P[0] = R.P[0]; rr.P[1] = R.P[1]; rr.P[2] = R.P[2];
    rr.blk = g.blk; rr.zs = zs; rr.as = n_out;
    res[i] = rr;
  };
  inc_machine(T, K, n, head, st, load, store);
  flush_inc_stats(cnt, st);
}

__global__ void __launch_bounds__(128) nonelastic_evap_kernel(Tables T, const Nucleus *nuc, uint64_t seed, uint64_t ev0, uint32_t n,
                                                              uint32_t *head, SecRec *slots, uint32_t *counts, const ResRec *res,
                                                              Counters *cnt) {
  unsigned long long c_bad = 0; double c_gam = 0;
  int ns = 0, zs = 0, as = 0;
  auto load = [&](uint32_t i, Residual &R, Rng &g) {
    const ResRec rr = res[i];
    g.init(seed, ev0 + i, 0u, rr.blk);
    R.Z = rr.Z; R.A = rr.A; R.estar = rr.estar; R.P[0] = rr.P[0]; R.P[1] = rr.P[1]; R.P[2] = rr.P[2]; R.mass_gs = nmass(T, rr.Z, rr.A);
    ns = (int)counts[i]; zs = rr.zs; as = rr.as;
  };
  auto emit = [&](uint32_t i, Rng &, const Emission &em) {
    SecRec rec{}; rec.Z = (int16_t)EJ_Z[em.j]; rec.A = (int16_t)EJ_A[em.j]; rec.origin = 1; rec.ke = em.ke;
    rec.dir[0] = em.dir.x; rec.dir[1] = em.dir.y; rec.dir[2] = em.dir.z;
    zs += rec.Z; as += rec.A;
    if (ns < MAX_SEC - 1) slots[(size_t)i * MAX_SEC + ns++] = rec; else atomicOr(&cnt->overflow, 128u);
  };
  auto done = [&](uint32_t i, Rng &, const Residual &R) {
    const double pn = sqrt(R.P[0] * R.P[0] + R.P[1] * R.P[1] + R.P[2] * R.P[2]);
    SecRec rec{}; rec.Z = (int16_t)R.Z; rec.A = (int16_t)R.A; rec.origin = 2; rec.ke = (float)residual_ke(R);
    if (pn > 0) { rec.dir[0] = (float)(R.P[0] / pn); rec.dir[1] = (float)(R.P[1] / pn); rec.dir[2] = (float)(R.P[2] / pn); }
    else { rec.dir[2] = 1.f; }
    zs += R.Z; as += R.A; slots[(size_t)i * MAX_SEC + ns++] = rec;
    if (zs != nuc->Z + 1 || as != nuc->A + 1) c_bad++;
    counts[i] = (uint32_t)ns; c_gam += R.estar;
  };
  evap_machine(T, n, head, load, emit, done);
  flush(&cnt->n_zab_bad, c_bad); flush(&cnt->e_gamma, c_gam);
}

// exclusive scan of counts[n] -> off[n+1] shifted by base (single block; n <= a few 1e5)
__global__ void __launch_bounds__(1024) scan_kernel(const uint32_t *counts, uint32_t n, uint32_t *off, unsigned long long *base_io) {
  __shared__ unsigned long long part[1024];
  const uint32_t per = (n + blockDim.x - 1) / blockDim.x, b = threadIdx.x * per, e = min(b + per, n);
  unsigned long long s = 0;
  for (uint32_t i = b; i < e; ++i) s += counts[i];
  part[threadIdx.x] = s; __syncthreads();
  if (threadIdx.x == 0) { unsigned long long acc = *base_io; for (int t = 0; t < (int)blockDim.x; ++t) { unsigned long long v = part[t]; part[t] = acc; acc += v; } *base_io = acc; }
  __syncthreads();
  unsigned long long acc = part[threadIdx.x];
  for (uint32_t i = b; i < e; ++i) { off[i] = (uint32_t)acc; acc += counts[i]; }
}
__global__ void __launch_bounds__(256) compact_kernel(const SecRec *slots, const uint32_t *counts, const uint32_t *off, uint32_t n,
                                                      SecRec *out, unsigned long long capacity) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t c = counts[i]; const unsigned long long o = off[i];
  for (uint32_t k = 0; k < c; ++k) if (o + k < capacity) out[o + k] = slots[(size_t)i * MAX_SEC + k];
}

// ------------------------------------------------------------------ sub-step test kernels
__global__ void philox_kernel(const uint32_t *in, uint64_t n, uint32_t *out) {
  const uint64_t i = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint4 r = philox4x32_10(make_uint4(in[6 * i], in[6 * i + 1], in[6 * i + 2], in[6 * i + 3]), make_uint2(in[6 * i + 4], in[6 * i + 5]));
  out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
}
__global__ void range_kernel(Tables T, int tab, const float *in, uint64_t n, float *out, int inverse) {
  const uint64_t i = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  if (!inverse) { const float x = logf(fminf(fmaxf(in[i], T.e_min), T.e_max)); out[i] = expf(ln_range(T, T.lnR, T.lnR2, tab, e_index(T, x))); }
  else out[i] = expf(ln_energy_of(T, T.lnE, T.lnE2, tab, logf(fmaxf(in[i], 1e-30f))));
}
__global__ void straggle_kernel(Tables T, float e, float mean, float rhoL, float zoa, uint64_t n, uint64_t seed, float *out) {
  const uint64_t i = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  Rng g; g.init(seed, i, 0u, 0u);
  const uint32_t spare = g.next4().x;
  out[i] = straggle(T, g, e, mean, rhoL, zoa, spare);
}

}  // namespace pmc
