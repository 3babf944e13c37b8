// oracle/opmc.cpp — fp64 CPU ORACLE for the proton Monte Carlo hot path of arxiv 1409.8336.
//
// TEST INFRASTRUCTURE ONLY (see opmc.h).  Plain, slow, one history at a time, written to be
// checked against PAPER.md by eye.  Shares no code with the CUDA path.  Citations are
// "PAPER.md:Lnn (§section)"; "Reading Rk" refers to the numbered list in DESIGN.md.
// Pins: tests/test_oracle_*.py.  Unpinned: see opmc.h header.
#include "opmc.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <string>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr double MP = 938.27208816, MN = 939.56542052, ME = 0.51099895;
constexpr double HBARC = 197.3269804;          // MeV fm
constexpr double KBETHE = 0.307075;            // MeV cm2/mol
constexpr double NAVO = 6.02214076e23;
constexpr double PI = 3.14159265358979323846;
constexpr double MEV_PER_G_TO_GY = 1.602176634e-10;
constexpr double INF = 1e300;

// ------------------------------------------------------------------ RNG (Reading R0)
// Philox4x32-10, Salmon et al.; key=(seed_lo,seed_hi), counter=(hist_lo,hist_hi,particle,block).
inline void philox(const uint32_t c_in[4], const uint32_t k_in[2], uint32_t out[4]) {
  uint32_t c0 = c_in[0], c1 = c_in[1], c2 = c_in[2], c3 = c_in[3], k0 = k_in[0], k1 = k_in[1];
  for (int r = 0; r < 10; ++r) {
    uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
    uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

struct Rng {
  uint32_t key[2], ctr[4], buf[4];
  int lane = 4;
  uint64_t ndraws = 0;
  Rng(uint64_t seed, uint64_t hist, uint32_t pid, uint32_t block0 = 0) {
    key[0] = (uint32_t)seed; key[1] = (uint32_t)(seed >> 32);
    ctr[0] = (uint32_t)hist; ctr[1] = (uint32_t)(hist >> 32); ctr[2] = pid; ctr[3] = block0;
  }
  uint32_t u32() {
    if (lane == 4) { philox(ctr, key, buf); ctr[3]++; lane = 0; }
    ndraws++;
    return buf[lane++];
  }
  double u() { return ((double)u32() + 0.5) * (1.0 / 4294967296.0); }   // in (0,1)
  double gauss() { double a = u(), b = u(); return std::sqrt(-2.0 * std::log(a)) * std::cos(2 * PI * b); }
  uint32_t child_id(uint32_t k) {   // Reading R0: id of the k-th product of this particle's event
    uint32_t c[4] = {ctr[0], ctr[1], ctr[2], (uint32_t)ndraws}, o[4];
    philox(c, key, o);
    return o[0] ^ (k + 1);
  }
};

// ------------------------------------------------------------------ small vector helpers
struct V3 { double x, y, z; };
inline V3 operator+(V3 a, V3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
inline V3 operator-(V3 a, V3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
inline V3 operator*(double s, V3 a) { return {s * a.x, s * a.y, s * a.z}; }
inline double dot(V3 a, V3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
inline double norm(V3 a) { return std::sqrt(dot(a, a)); }
inline V3 unit(V3 a) { double n = norm(a); return {a.x / n, a.y / n, a.z / n}; }
inline V3 cross(V3 a, V3 b) { return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x}; }

// components (a,b,c) given in the frame whose z axis is the unit vector d -> lab frame
inline V3 to_lab(V3 d, double a, double b, double c) {
  double s2 = d.x * d.x + d.y * d.y;
  if (s2 < 1e-20) { double sg = d.z >= 0 ? 1.0 : -1.0; return {a, sg * b, sg * c}; }
  double s = std::sqrt(s2);
  V3 e1{d.x * d.z / s, d.y * d.z / s, -s}, e2{-d.y / s, d.x / s, 0.0};
  return a * e1 + b * e2 + c * d;
}
inline V3 isotropic(Rng &g) {
  double c = 2 * g.u() - 1, ph = 2 * PI * g.u(), s = std::sqrt(std::max(0.0, 1 - c * c));
  return {s * std::cos(ph), s * std::sin(ph), c};
}
// Lorentz transformation of (p,E) from a frame moving with velocity beta (seen from the target frame)
inline void boost(V3 beta, V3 &p, double &E) {
  double b2 = dot(beta, beta);
  if (b2 <= 0) return;
  double gam = 1.0 / std::sqrt(1.0 - b2), bp = dot(beta, p);
  double f = (gam - 1.0) * bp / b2 + gam * E;
  p = p + f * beta;
  E = gam * (E + bp);
}

// ------------------------------------------------------------------ Cugnon NN parameterisation
// PAPER.md:L77 ref [20]; formulas = Reading R6.  p in GeV/c, sigma in mb.
double cug_sigma_pp(double p) {
  if (p < 0.44) return 34.0 * std::pow(p / 0.4, -2.104);
  if (p < 0.8) return 23.5 + 1000.0 * std::pow(p - 0.7, 4);
  if (p < 2.0) return 1250.0 / (p + 50.0) - 4.0 * (p - 1.3) * (p - 1.3);
  return 77.0 / (p + 1.5);
}
double cug_sigma_np(double p) {
  if (p < 0.446) { double l = std::log(p); return 6.3555 * std::pow(p, -3.2481) * std::exp(-0.377 * l * l); }
  if (p < 0.8) return 33.0 + 196.0 * std::pow(std::fabs(p - 0.95), 2.5);
  if (p < 2.0) return 31.0 / std::sqrt(p);
  return 77.0 / (p + 1.5);
}
double cug_b_pp(double p) { if (p < 2.0) { double p8 = std::pow(p, 8); return 5.5 * p8 / (7.7 + p8); } return 5.334 + 0.67 * (p - 2.0); }
double cug_b_np(double p) {
  if (p < 0.225) return 0.0;
  if (p < 0.6) return 16.53 * (p - 0.225);
  if (p < 1.6) return -1.63 * p + 7.16;
  return cug_b_pp(p);
}
double cug_a_np(double p) { return p < 0.8 ? 1.0 : 0.64 / (p * p); }

// cos(theta_cm) of NN elastic scattering: dsigma/dt ~ exp(B t) (+ a exp(B u) for np)
double sample_nn_cos(Rng &g, bool same_type, double p_lab_gev, double pcm_mev) {
  double tmax = 4.0 * pcm_mev * pcm_mev * 1e-6;          // (GeV/c)^2
  double B = same_type ? cug_b_pp(p_lab_gev) : cug_b_np(p_lab_gev);
  bool backward = false;
  if (!same_type) { double a = cug_a_np(p_lab_gev); backward = g.u() < a / (1.0 + a); }
  double u = g.u(), t;
  if (B * tmax < 1e-9) t = u * tmax;
  else t = -std::log(1.0 - u * (1.0 - std::exp(-B * tmax))) / B;
  double c = 1.0 - 2.0 * t / tmax;
  return backward ? -c : c;
}

// ------------------------------------------------------------------ tables
struct Tables {
  int n_e = 0, n_sr = 0, n_r = 0, n_elem = 0, zdim = 0, adim = 0;
  double e_min = 0, e_max = 0, dlne = 0;
  std::vector<double> stop, lnR, lnR2, lnRlo, lnRhi, lnE, lnE2, sne, sel, mass, ek, ec;
  std::vector<int> ez, ea;
  double e_cut = 0.1, highland = 1.07, kappa_g = 10, s_max = 0.2;
  int n_batches = 10;
  std::vector<double> mol_c0, mol_c1, mol_c2; double mol_dth = 0;      // Moliere tables (Reading R12)
  bool loaded = false;

  static double spline(const double *y, const double *y2, int n, double x0, double h, double x) {
    // natural cubic spline on uniform knots ("second derivatives are also precalculated")
    double t = (x - x0) / h;
    int i = (int)std::floor(t);
    if (i < 0) i = 0;
    if (i > n - 2) i = n - 2;
    double b = t - i, a = 1.0 - b;
    return a * y[i] + b * y[i + 1] + ((a * a * a - a) * y2[i] + (b * b * b - b) * y2[i + 1]) * h * h / 6.0;
  }
  double range_gcm2(int t, double e) const {       // CSDA range of table t at energy e
    double x = std::log(std::min(std::max(e, e_min), e_max));
    return std::exp(spline(&lnR[t * n_e], &lnR2[t * n_e], n_e, std::log(e_min), dlne, x));
  }
  double energy_of_range(int t, double r) const {  // inverse table
    double lo = lnRlo[t], hi = lnRhi[t], x = std::log(std::max(r, 1e-300));
    if (x <= lo) return e_min;
    if (x >= hi) return e_max;
    double h = (hi - lo) / (n_r - 1);
    return std::exp(spline(&lnE[t * n_r], &lnE2[t * n_r], n_r, lo, h, x));
  }
  double sigma(const std::vector<double> &tab, int el, double e) const {   // linear in ln E (Reading R5)
    double t = (std::log(std::min(std::max(e, e_min), e_max)) - std::log(e_min)) / dlne;
    int i = std::min(std::max((int)std::floor(t), 0), n_e - 2);
    double b = t - i;
    return (1 - b) * tab[el * n_e + i] + b * tab[el * n_e + i + 1];
  }
  double nmass(int z, int a) const { return (z < 0 || a < 1 || z >= zdim || a >= adim || z > a) ? 0.0 : mass[z * adim + a]; }
};

struct Material {
  int hu_lo, hu_hi; double rho_lo, rho_hi, w[OPMC_MAX_ELEM], f_m, x0; int table_id;
  double zoa;                                   // <Z/A> = sum w_i Z_i/A_i
};

// ------------------------------------------------------------------ nucleus model (Reading R6.1)
constexpr int NSHELL_MAX = 15;
struct Nucleus {
  int Z = 0, A = 0, nshell = 15;
  double rmax = 0, rout[NSHELL_MAX], rho[2][NSHELL_MAX], pF[2][NSHELL_MAX], EF[2][NSHELL_MAX], V[2][NSHELL_MAX];
  double coulomb = 0;                           // B_C for protons
  bool pauli = true; double const_sigma_mb = -1;  // test switches (closed-form pin only)
  long step_guard = 1024;                       // Reading R6.8; option "inc_step_guard" (pin test of the guard only)
};
inline double nucleon_mass(int type) { return type == 0 ? MP : MN; }   // type 0 = proton, 1 = neutron

Nucleus build_nucleus(const Tables &T, int Z, int A) {
  // Woods-Saxon approximated by 15 constant-density shells, two-component Fermi gas.
  Nucleus n; n.Z = Z; n.A = A; n.nshell = 15;
  double c = 1.07 * std::cbrt((double)A), a = 0.545;
  n.rmax = c + a * std::log(99.0);
  double dr = n.rmax / 15, vol[15], avg[15], tot = 0;
  for (int k = 0; k < 15; ++k) {
    double r0 = k * dr, r1 = (k + 1) * dr, num = 0;
    const int M = 200;
    for (int i = 0; i < M; ++i) { double r = r0 + (i + 0.5) * dr / M; num += r * r / (1.0 + std::exp((r - c) / a)) * dr / M; }
    vol[k] = 4 * PI / 3 * (r1 * r1 * r1 - r0 * r0 * r0);
    avg[k] = 4 * PI * num / vol[k];
    tot += avg[k] * vol[k];
    n.rout[k] = r1;
  }
  double sep[2];
  sep[0] = T.nmass(Z - 1, A - 1) + MP - T.nmass(Z, A);
  sep[1] = T.nmass(Z, A - 1) + MN - T.nmass(Z, A);
  for (int k = 0; k < 15; ++k) {
    double rho = avg[k] * A / tot;
    for (int t = 0; t < 2; ++t) {
      double frac = t == 0 ? (double)Z / A : (double)(A - Z) / A, m = nucleon_mass(t);
      n.rho[t][k] = rho * frac;
      n.pF[t][k] = HBARC * std::cbrt(3 * PI * PI * n.rho[t][k]);
      n.EF[t][k] = std::sqrt(n.pF[t][k] * n.pF[t][k] + m * m) - m;      // Reading R6.1b: relativistic E_F
      n.V[t][k] = n.EF[t][k] + sep[t];
    }
  }
  n.coulomb = 1.44 * (Z - 1) / n.rmax;
  return n;
}

struct Sec { int Z, A, origin; double ke; V3 dir; };
struct Residual { int Z, A; double estar; V3 P; double mass_gs; };

struct EventCheck {
  double max_resid = 0; uint64_t zab_bad = 0; uint64_t inc_tries = 0;
  // how often the limits of Reading R6.8 end an attempt, and how deep a cascade gets (bookkeeping only)
  uint64_t guard_trips = 0, stack_trips = 0, max_stack = 0, max_out = 0;
};

// ------------------------------------------------------------------ INC (Reading R6)
struct CascNucleon { int type; V3 r, p; int shell; };

// one attempt; returns false if no Pauli-allowed collision happened or the outcome is invalid
bool inc_attempt(const Tables &T, const Nucleus &N, double t_in, Rng &g, std::vector<Sec> &out, Residual &res,
                 EventCheck *chk = nullptr) {
  out.clear();
  const int ns = N.nshell;
  // entry: uniform over the disc of radius rmax, travelling along +z (L75 "random point of entry")
  double b = N.rmax * std::sqrt(g.u()), ph = 2 * PI * g.u();
  V3 r{b * std::cos(ph), b * std::sin(ph), -std::sqrt(std::max(0.0, N.rmax * N.rmax - b * b))};
  V3 dir{0, 0, 1};
  std::vector<CascNucleon> stack;
  int ncoll = 0;
  {  // refraction into the outermost shell: gains V (tangential momentum conserved)
    double Tn = t_in + N.V[0][ns - 1], p0 = std::sqrt(t_in * (t_in + 2 * MP)), p1 = std::sqrt(Tn * (Tn + 2 * MP));
    V3 nh = unit(r); V3 pv = p0 * dir; double pr = dot(pv, nh); V3 pt = pv - pr * nh;
    double pr2 = p1 * p1 - dot(pt, pt);
    V3 pnew = pt + (-std::sqrt(std::max(pr2, 0.0))) * nh;
    stack.push_back({0, r, pnew, ns - 1});
  }
  double e_out_sum = 0; V3 p_out_sum{0, 0, 0}; int n_out = 0, np_out = 0;
  long guard = 0;
  while (!stack.empty()) {
    CascNucleon c = stack.back(); stack.pop_back();
    bool alive = true;
    while (alive) {
      if (++guard > N.step_guard) { if (chk) chk->guard_trips++; return false; }   // Reading R6.8: a nucleon on a bound orbit in a dilute shell never ends the attempt
      int k = c.shell, ty = c.type;
      double m = nucleon_mass(ty), p2 = dot(c.p, c.p), E = std::sqrt(p2 + m * m), Tk = E - m;
      V3 d = (1.0 / std::sqrt(p2)) * c.p;
      // candidate collisions with a proton and with a neutron of the Fermi sea (Reading R6.3)
      double dbest = INF; int tbest = -1; V3 qbest{0, 0, 0}; double plab_best = 0;
      for (int tp = 0; tp < 2; ++tp) {
        if (N.rho[tp][k] <= 0) continue;
        double mq = nucleon_mass(tp);
        double qmag = N.pF[tp][k] * std::cbrt(g.u());
        V3 q = qmag * isotropic(g);
        double Eq = std::sqrt(qmag * qmag + mq * mq);
        V3 Pt = c.p + q; double s = (E + Eq) * (E + Eq) - dot(Pt, Pt);
        double e1 = (s - m * m - mq * mq) / (2 * mq), plab = std::sqrt(std::max(e1 * e1 - m * m, 0.0));
        double sig = N.const_sigma_mb >= 0 ? N.const_sigma_mb
                                           : (tp == ty ? cug_sigma_pp(plab * 1e-3) : cug_sigma_np(plab * 1e-3));
        double dist = -std::log(g.u()) / (N.rho[tp][k] * sig * 0.1);     // 1 mb = 0.1 fm^2
        if (dist < dbest) { dbest = dist; tbest = tp; qbest = q; plab_best = plab; }
      }
      // distance to the shell boundaries along d
      double rr = dot(c.r, c.r), bq = dot(c.r, d), r_out = N.rout[k], r_in = k > 0 ? N.rout[k - 1] : 0.0;
      double dbound = -bq + std::sqrt(std::max(bq * bq - (rr - r_out * r_out), 0.0)); bool inward = false;
      if (k > 0 && bq < 0) {
        double disc = bq * bq - (rr - r_in * r_in);
        if (disc > 0) { double s_in = -bq - std::sqrt(disc); if (s_in < dbound) { dbound = std::max(s_in, 0.0); inward = true; } }
      }
      if (dbest < dbound) {
        // ---- collision attempt (Reading R6.4)
        c.r = c.r + dbest * d;
        int tp = tbest; double mq = nucleon_mass(tp);
        V3 q = qbest; double Eq = std::sqrt(dot(q, q) + mq * mq);
        V3 Pt = c.p + q; double Et = E + Eq; V3 beta = (1.0 / Et) * Pt;
        double s = Et * Et - dot(Pt, Pt);
        double pcm = std::sqrt(std::max((s - (m + mq) * (m + mq)) * (s - (m - mq) * (m - mq)), 0.0) / (4 * s));
        V3 p1 = c.p; double E1 = E; boost(-1.0 * beta, p1, E1);        // projectile in the CM
        V3 ax = unit(p1);
        double ct = sample_nn_cos(g, tp == ty, plab_best * 1e-3, pcm), st = std::sqrt(std::max(0.0, 1 - ct * ct));
        double phi = 2 * PI * g.u();
        V3 n1 = pcm * to_lab(ax, st * std::cos(phi), st * std::sin(phi), ct), n2 = -1.0 * n1;
        double En1 = std::sqrt(pcm * pcm + m * m), En2 = std::sqrt(pcm * pcm + mq * mq);
        boost(beta, n1, En1); boost(beta, n2, En2);
        double T1 = En1 - m, T2 = En2 - mq;
        bool ok = !N.pauli || (T1 > N.EF[ty][k] && T2 > N.EF[tp][k]);   // L77 Pauli blocking
        if (!ok) continue;                                              // blocked: go on unchanged
        ncoll++;
        // trapping (Reading R6.4): outside energy eps = T - V <= B_C stays in the nucleus
        double bc2 = tp == 0 ? N.coulomb : 0.0, bc1 = ty == 0 ? N.coulomb : 0.0;
        if (T2 - N.V[tp][k] > bc2) stack.push_back({tp, c.r, n2, k});
        if (T1 - N.V[ty][k] > bc1) { c.p = n1; } else alive = false;
        if (chk) chk->max_stack = std::max<uint64_t>(chk->max_stack, stack.size());
        if ((int)stack.size() > 200) { if (chk) chk->stack_trips++; return false; }
        continue;
      }
      // ---- shell boundary (L77 "reflection and refraction", Reading R6.5)
      c.r = c.r + dbound * d;
      double rb = inward ? r_in : r_out;
      c.r = (rb / norm(c.r)) * c.r;
      V3 nh = (1.0 / rb) * c.r;
      double pr = dot(c.p, nh); V3 pt = c.p - pr * nh;
      int k2 = inward ? k - 1 : k + 1;
      double Vnew = k2 >= ns ? 0.0 : N.V[ty][k2], T2 = Tk + (Vnew - N.V[ty][k]);
      double pn2 = T2 > 0 ? T2 * (T2 + 2 * m) : -1.0, pr2 = pn2 - dot(pt, pt);
      if (pn2 <= 0 || pr2 <= 0) { c.p = pt - pr * nh; continue; }       // specular reflection
      V3 pnew = pt + ((pr > 0 ? 1.0 : -1.0) * std::sqrt(pr2)) * nh;
      if (k2 >= ns) {                                                  // leaves the nucleus with KE = eps
        out.push_back({ty == 0 ? 1 : 0, 1, 0, T2, unit(pnew)});
        e_out_sum += T2 + m; p_out_sum = p_out_sum + pnew; n_out++; if (ty == 0) np_out++;
        alive = false;
      } else { c.p = pnew; c.shell = k2; }
    }
  }
  if (chk) chk->max_out = std::max<uint64_t>(chk->max_out, (uint64_t)n_out);
  if (ncoll == 0) return false;                                        // L75: need >= 1 allowed collision
  // ---- residual nucleus (Reading R6.7): exact integers, relativistic invariant mass
  int Ar = N.A + 1 - n_out, Zr = N.Z + 1 - np_out;
  double Mt = T.nmass(N.Z, N.A), Mgs = T.nmass(Zr, Ar);
  if (Ar < 1 || Zr < 0 || Zr > Ar || Mgs <= 0) return false;
  double pin = std::sqrt(t_in * (t_in + 2 * MP));
  double Eres = (t_in + MP + Mt) - e_out_sum; V3 Pres = V3{0, 0, pin} - p_out_sum;
  double M2 = Eres * Eres - dot(Pres, Pres);
  if (Eres <= 0 || M2 <= 0) return false;
  double estar = std::sqrt(M2) - Mgs;
  if (estar < 0) return false;
  if (Ar == 1 && estar > 1e-9) return false;                           // a lone nucleon cannot be excited
  res = {Zr, Ar, estar, Pres, Mgs};
  return true;
}

void inc_event(const Tables &T, const Nucleus &N, double t_in, Rng &g, std::vector<Sec> &out, Residual &res, EventCheck &chk) {
  for (int tries = 0; tries < 100000; ++tries) {   // L75 "This is repeated until ..."
    chk.inc_tries++;
    if (inc_attempt(T, N, t_in, g, out, res, &chk)) return;
  }
  // Reading R6.8 (never reached in the configs): give up and form the compound nucleus (Z+1, A+1)
  out.clear();
  double pin = std::sqrt(t_in * (t_in + 2 * MP)), Et = t_in + MP + T.nmass(N.Z, N.A), Mgs = T.nmass(N.Z + 1, N.A + 1);
  res = {N.Z + 1, N.A + 1, std::sqrt(Et * Et - pin * pin) - Mgs, V3{0, 0, pin}, Mgs};
}

// ------------------------------------------------------------------ evaporation (Reading R7)
constexpr int EJ_Z[6] = {0, 1, 1, 1, 2, 2}, EJ_A[6] = {1, 1, 2, 3, 3, 4};
constexpr double EJ_SPIN_G[6] = {2, 2, 3, 2, 2, 1};
constexpr int NQ = 64;
inline double pairing(int Z, int A) { int N = A - Z; double d = 12.0 / std::sqrt((double)A); return (Z % 2 == 0 && N % 2 == 0) ? 2 * d : ((Z % 2) != (N % 2) ? d : 0.0); }

struct Channel { bool open = false; double S = 0, emin = 0, emax = 0, width = 0, f[NQ]; int Zd = 0, Ad = 0; };

void evap_channels(const Tables &T, int Z, int A, double estar, uint32_t mask, Channel ch[6]) {
  double ref = 2.0 * std::sqrt(A / 8.0 * std::max(estar, 0.0));
  double Mpar = T.nmass(Z, A);
  for (int j = 0; j < 6; ++j) {
    Channel &c = ch[j]; c = Channel();
    if (!((mask >> j) & 1)) continue;
    int Zd = Z - EJ_Z[j], Ad = A - EJ_A[j];
    if (Ad < 2 || Zd < 0) continue;
    double Md = T.nmass(Zd, Ad), mj = T.nmass(EJ_Z[j], EJ_A[j]);
    if (Md <= 0) continue;
    c.Zd = Zd; c.Ad = Ad; c.S = Md + mj - Mpar;
    double a13 = std::cbrt((double)Ad), kV = 0, cj = 0;
    if (j > 0) {
      double rhoj = j == 1 ? 0.0 : 1.2, V = 1.44 * EJ_Z[j] * Zd / (1.5 * a13 + rhoj);
      kV = T.ek[j * T.zdim + Zd] * V; cj = T.ec[j * T.zdim + Zd];
    }
    c.emin = kV; c.emax = estar - c.S - pairing(Zd, Ad);
    if (c.emax <= c.emin) continue;
    double alpha = 0.76 + 2.2 / a13, beta = (2.12 / (a13 * a13) - 0.050) / alpha, ad = Ad / 8.0;
    double gj = EJ_SPIN_G[j] * mj, de = (c.emax - c.emin) / NQ, geo = a13 * a13;
    for (int i = 0; i < NQ; ++i) {
      double e = c.emin + (i + 0.5) * de;
      double sinv = j == 0 ? geo * alpha * (1 + beta / e) : geo * (1 + cj) * (1 - kV / e);
      c.f[i] = gj * sinv * e * std::exp(2.0 * std::sqrt(ad * (c.emax - e)) - ref);
      c.width += c.f[i] * de;
    }
    c.open = c.width > 0;
  }
}

// one emission; returns channel index or -1 if nothing can be emitted
int evap_emit(const Tables &T, Residual &R, Rng &g, uint32_t mask, Sec &sec, double *eps_out, double *cos_out) {
  Channel ch[6];
  evap_channels(T, R.Z, R.A, R.estar, mask, ch);
  double tot = 0; for (int j = 0; j < 6; ++j) if (ch[j].open) tot += ch[j].width;
  if (tot <= 0) return -1;
  double u = g.u() * tot; int j = -1;
  for (int q = 0; q < 6; ++q) if (ch[q].open) { j = q; if (u < ch[q].width) break; u -= ch[q].width; }
  Channel &c = ch[j];
  double de = (c.emax - c.emin) / NQ, v = g.u() * c.width / de; int bin = NQ - 1;
  for (int i = 0; i < NQ; ++i) { if (v < c.f[i]) { bin = i; break; } v -= c.f[i]; }
  double eps = c.emin + (bin + g.u()) * de;                             // total CM kinetic energy released
  // relativistic two-body decay of M* -> m_j + M_d* (isotropic in the nucleus rest frame, L79)
  double mj = T.nmass(EJ_Z[j], EJ_A[j]), Mdgs = T.nmass(c.Zd, c.Ad);
  double Mstar = R.mass_gs + R.estar, Ud = R.estar - c.S - eps, Md = Mdgs + Ud;
  double pc2 = (Mstar * Mstar - (mj + Md) * (mj + Md)) * (Mstar * Mstar - (mj - Md) * (mj - Md)) / (4 * Mstar * Mstar);
  double pc = std::sqrt(std::max(pc2, 0.0));
  V3 dirc = isotropic(g);
  V3 pj = pc * dirc, pd = -1.0 * pj; double Ej = std::sqrt(pc * pc + mj * mj), Ed = std::sqrt(pc * pc + Md * Md);
  double Epar = std::sqrt(dot(R.P, R.P) + Mstar * Mstar); V3 beta = (1.0 / Epar) * R.P;
  boost(beta, pj, Ej); boost(beta, pd, Ed);
  sec = {EJ_Z[j], EJ_A[j], 1, Ej - mj, norm(pj) > 0 ? unit(pj) : V3{0, 0, 1}};
  R = {c.Zd, c.Ad, Ud, pd, Mdgs};
  if (eps_out) *eps_out = eps;
  if (cos_out) *cos_out = dirc.z;
  return j;
}

void evaporate(const Tables &T, Residual &R, Rng &g, std::vector<Sec> &out) {
  for (int it = 0; it < 200; ++it) { Sec s; if (evap_emit(T, R, g, 0x3F, s, nullptr, nullptr) < 0) break; out.push_back(s); }
}

// full non-elastic event in the frame where the proton moves along +z; checks conservation
void nonelastic_event(const Tables &T, const Nucleus &N, double t_in, Rng &g, std::vector<Sec> &secs, Residual &R,
                      EventCheck &chk) {
  inc_event(T, N, t_in, g, secs, R, chk);
  evaporate(T, R, g, secs);
  // conservation audit (north_star: charge and baryon number exact; 4-momentum to rounding)
  int zs = R.Z, as = R.A; double Mres = R.mass_gs + R.estar;
  double Es = std::sqrt(dot(R.P, R.P) + Mres * Mres); V3 Ps = R.P;
  for (const Sec &s : secs) {
    zs += s.Z; as += s.A; double m = T.nmass(s.Z, s.A), p = std::sqrt(s.ke * (s.ke + 2 * m));
    Es += s.ke + m; Ps = Ps + p * s.dir;
  }
  if (zs != N.Z + 1 || as != N.A + 1) chk.zab_bad++;
  double pin = std::sqrt(t_in * (t_in + 2 * MP));
  double r = std::max(std::fabs(Es - (t_in + MP + T.nmass(N.Z, N.A))), norm(Ps - V3{0, 0, pin}));
  chk.max_resid = std::max(chk.max_resid, r);
}

// ------------------------------------------------------------------ nuclear elastic (Eq.3, Reading R5)
struct ElasticOut { double t_gev2, T_out, T_rec; V3 dir_out, dir_rec; };
ElasticOut elastic_event(const Tables &T, int Z, int A, double Tk, Rng &g, EventCheck &chk) {
  double M = T.nmass(Z, A), E = Tk + MP, plab = std::sqrt(Tk * (Tk + 2 * MP));
  double s = MP * MP + M * M + 2 * M * E, rs = std::sqrt(s), pcm = M * plab / rs;
  double tmax = 4 * pcm * pcm * 1e-6, ct;
  if (A == 1) {
    ct = sample_nn_cos(g, true, plab * 1e-3, pcm);                      // p-p: Cugnon angular law
  } else {
    double a1, b1, a2, b2, Ad = A;
    if (A <= 62) { a1 = std::pow(Ad, 1.63); b1 = 14.5 * std::pow(Ad, 0.66); a2 = 1.4 * std::pow(Ad, 0.33); b2 = 10; }
    else { a1 = std::pow(Ad, 1.33); b1 = 60 * std::pow(Ad, 0.33); a2 = 0.4 * std::pow(Ad, 0.4); b2 = 10; }
    double w1 = a1 * (1 - std::exp(-b1 * tmax)) / b1, w2 = a2 * (1 - std::exp(-b2 * tmax)) / b2;
    double bb = g.u() * (w1 + w2) < w1 ? b1 : b2;
    double t = -std::log(1 - g.u() * (1 - std::exp(-bb * tmax))) / bb;  // |t|, truncated exponential
    ct = 1 - 2 * t / tmax;
  }
  double phi = 2 * PI * g.u(), st = std::sqrt(std::max(0.0, 1 - ct * ct));
  V3 pc{pcm * st * std::cos(phi), pcm * st * std::sin(phi), pcm * ct};
  V3 pr = -1.0 * pc; double Ep = std::sqrt(pcm * pcm + MP * MP), Er = std::sqrt(pcm * pcm + M * M);
  V3 beta{0, 0, plab / (E + M)};
  boost(beta, pc, Ep); boost(beta, pr, Er);
  ElasticOut o; o.t_gev2 = 0.5 * tmax * (1 - ct); o.T_out = Ep - MP; o.T_rec = Er - M;
  o.dir_out = unit(pc); o.dir_rec = norm(pr) > 0 ? unit(pr) : V3{0, 0, 1};
  chk.max_resid = std::max(chk.max_resid, std::max(std::fabs(o.T_out + o.T_rec - Tk), norm(pc + pr - V3{0, 0, plab})));
  return o;
}

// ------------------------------------------------------------------ straggling (Reading R4)
double straggle(const Tables &T, Rng &g, double e_start, double mean_loss, double rhoL, double zoa) {
  if (rhoL <= 0 || mean_loss <= 0) return mean_loss;
  double gam = 1 + e_start / MP, b2 = 1 - 1 / (gam * gam), bg2 = b2 * gam * gam;
  double tmax = 2 * ME * bg2 / (1 + 2 * gam * ME / MP + (ME / MP) * (ME / MP));
  double xi = 0.5 * KBETHE * zoa * rhoL / b2, kappa = xi / tmax, loss;
  if (kappa >= T.kappa_g) {
    loss = mean_loss + std::sqrt(xi * tmax * (1 - 0.5 * b2)) * g.gauss();
  } else {
    // Vavilov as its defining compound-Poisson process; collisions below T_c lumped into a Gaussian
    double tc = std::min(1e-3, tmax / 100);
    double mu = xi * ((1 / tc - 1 / tmax) - b2 / tmax * std::log(tmax / tc));
    double mean_hard = xi * (std::log(tmax / tc) - b2 * (1 - tc / tmax));
    double hard = 0, acc = -std::log(g.u());
    while (acc < mu) {
      double t;
      do { t = 1.0 / (1 / tc - g.u() * (1 / tc - 1 / tmax)); } while (g.u() >= 1 - b2 * t / tmax);
      hard += t; acc += -std::log(g.u());
    }
    double var_soft = xi * tc * (1 - b2 * tc / (2 * tmax));
    loss = mean_loss + (hard - mean_hard) + std::sqrt(var_soft) * g.gauss();
  }
  return std::min(std::max(loss, 0.0), e_start);
}

}  // namespace

// =============================================================================================
struct opmc_ctx {
  Tables T;
  std::vector<Material> mats;
  std::vector<Nucleus> nuc;                   // per element (A > 1)
  std::vector<int16_t> hu; int nx = 0, ny = 0, nz = 0; double d[3] = {0, 0, 0}, org[3] = {0, 0, 0};
  bool opt_strag = true, opt_mcs = true, opt_el = true, opt_ne = true; int threads = 0;
  // per-spot dose influence on a list of ROI voxels (Reading R11)
  std::vector<int32_t> roi_vox, roi_map; std::vector<double> dij; int dij_spots = 0;
  int mcs_model = 0;                          // 0 Highland x 1.07 (the paper's results), 1 full Moliere (L59; Reading R12)
  bool score_let = false; std::vector<double> let_num, let_den;   // LET_d tallies (Reading R9)
  long inc_step_guard = 1024;                 // Reading R6.8 (option "inc_step_guard": pin test of the guard only)
  uint64_t ev_el[OPMC_MAX_ELEM] = {0}, ev_ne[OPMC_MAX_ELEM] = {0};   // events per class and target element (pin test bookkeeping)
  opmc_counters cnt{};
  std::string err;
};

namespace {

struct Particle { V3 r, d; double E; int idx[3]; uint32_t pid; uint32_t block0; int spot = 0; };
struct Ledger { double dep = 0, esc = 0, neu = 0, gam = 0, q = 0, air = 0; };

const Material &material_of(const opmc_ctx *c, int hu) {
  for (const Material &m : c->mats) if (hu >= m.hu_lo && hu < m.hu_hi) return m;
  return hu < c->mats.front().hu_lo ? c->mats.front() : c->mats.back();     // clamp (L49: >3060 -> Ti)
}
inline double density(const Material &m, int hu) {
  int h = std::min(std::max(hu, m.hu_lo), m.hu_hi);
  return m.rho_lo + (m.rho_hi - m.rho_lo) * (double)(h - m.hu_lo) / (double)(m.hu_hi - m.hu_lo);
}
// water-equivalent factor: g/cm2 of the material's table per cm of path (Eq.1/Eq.2)
inline double wet_factor(const Material &m, double rho) { return m.table_id == 0 ? rho * m.f_m : rho; }

double sigma_macro(const opmc_ctx *c, const Material &m, double rho, double e, bool el, bool ne, double *per_elem_el,
                   double *per_elem_ne) {
  double tot = 0;
  for (int i = 0; i < c->T.n_elem; ++i) {
    double n_i = rho * NAVO * m.w[i] / c->T.ea[i] * 1e-27;                  // per (cm * mb)
    double a = el ? n_i * c->T.sigma(c->T.sel, i, e) : 0.0, b = ne ? n_i * c->T.sigma(c->T.sne, i, e) : 0.0;
    if (per_elem_el) per_elem_el[i] = a;
    if (per_elem_ne) per_elem_ne[i] = b;
    tot += a + b;
  }
  return tot;
}

// distance along d from r to the first face of voxel idx; axis_out = which face
double dist_to_face(const opmc_ctx *c, const V3 &r, const V3 &d, const int idx[3], int &axis, int &sgn) {
  const double rr[3] = {r.x, r.y, r.z}, dd[3] = {d.x, d.y, d.z};
  double best = INF; axis = -1; sgn = 0;
  for (int a = 0; a < 3; ++a) {
    if (dd[a] == 0) continue;
    double face = dd[a] > 0 ? (idx[a] + 1) * c->d[a] : idx[a] * c->d[a];
    double t = std::max((face - rr[a]) / dd[a], 0.0);
    if (t < best) { best = t; axis = a; sgn = dd[a] > 0 ? 1 : -1; }       // ties: x before y before z
  }
  return best;
}

// one MCS deflection of width theta0 (two independent projected Gaussians), Reading R3.4
inline V3 deflect(Rng &g, V3 d, double theta0) {
  double th = theta0 * std::sqrt(-2 * std::log(g.u())), ph = 2 * PI * g.u();
  return unit(to_lab(d, std::sin(th) * std::cos(ph), std::sin(th) * std::sin(ph), std::cos(th)));
}
inline double highland(const Tables &T, double e, double rhoL, double x0) {
  if (rhoL <= 0) return 0;
  double pc = std::sqrt(e * (e + 2 * MP)), bcp = pc * pc / (e + MP), t = rhoL / x0;
  return T.highland * 13.6 / bcp * std::sqrt(t) * std::max(0.0, 1 + 0.038 * std::log(t));
}

// energy e (MeV) deposited in voxel vox by a history of spot `spot` -> row spot, column roi_map[vox] of the influence matrix
inline void score_influence(opmc_ctx *c, int spot, size_t vox, double e) {
  if (c->roi_map.empty() || e == 0) return;
  const int32_t j = c->roi_map[vox];
  if (j < 0) return;
  #pragma omp atomic
  c->dij[(size_t)spot * c->roi_vox.size() + j] += e;
}

// Full Moliere theory (Bethe 1953; Reading R12).  Space angle after mass thickness t = rho dx of a mixture:
//   chi_c^2 = 0.157 t sum_i w_i Z_i(Z_i+1)/A_i / (p beta)^2,   chi_a,i^2 = 2.007e-5 Z_i^(2/3) [1 + 3.34 (Z_i alpha/beta)^2] / p^2,
//   ln chi_a^2 = Z(Z+1)/A-weighted mean of ln chi_a,i^2,  b = ln(chi_c^2/chi_a^2) + 1 - 2 C_Euler,  B - ln B = b,
//   f(theta) theta dtheta = x dx [2 e^{-x^2} + f1(x)/B + f2(x)/B^2],  x = theta / (chi_c sqrt(B)).
// x is drawn by inverting the tabulated cumulative C0 + C1/B + C2/B^2 (uniform in x^2 inside a bin), beyond the table
// from the single-scattering tail 1/(B x^2).  Fewer than 20 collisions (Omega < 20): outside the theory -> Highland.
inline bool moliere_angle(const opmc_ctx *c, const Material &m, double rho, double e, double dx, Rng &g, double &theta) {
  const Tables &T = c->T;
  const double p2 = e * (e + 2 * MP), E = e + MP, beta2 = p2 / (E * E), pb = p2 / E, t = dx * rho;
  double zs = 0, zl = 0;
  for (int i = 0; i < T.n_elem; ++i) {
    if (m.w[i] <= 0) continue;
    const double Z = T.ez[i], q = m.w[i] * Z * (Z + 1) / T.ea[i];
    const double za = Z / 137.035999 , chia2 = 2.007e-5 * std::pow(Z, 2.0 / 3.0) * (1 + 3.34 * za * za / beta2) / p2;
    zs += q; zl += q * std::log(chia2);
  }
  if (zs <= 0 || t <= 0) return false;
  const double chic2 = 0.157 * zs * t / (pb * pb), ln_omega = std::log(chic2) - zl / zs;
  if (ln_omega < std::log(20.0)) return false;
  const double b = ln_omega + 1 - 2 * 0.5772156649015329;
  double B = b + std::log(b);
  for (int it = 0; it < 8; ++it) B -= (B - std::log(B) - b) / (1 - 1 / B);
  const int n = (int)T.mol_c0.size(); const double dth = T.mol_dth, xmax = (n - 1) * dth;
  auto C = [&](int k) { return T.mol_c0[k] + T.mol_c1[k] / B + T.mol_c2[k] / (B * B); };
  const double tail = 1 / (B * xmax * xmax), total = C(n - 1) + tail, U = g.u() * total;
  double x;
  if (U >= C(n - 1)) x = 1 / std::sqrt(B * std::max(total - U, 1e-300));
  else {
    int k = 0;
    while (k < n - 2 && C(k + 1) <= U) ++k;
    const double c0 = C(k), c1 = C(k + 1), f = c1 > c0 ? std::min(std::max((U - c0) / (c1 - c0), 0.0), 1.0) : 0.5;
    const double x0 = k * dth, x1 = (k + 1) * dth;
    x = std::sqrt(x0 * x0 + f * (x1 * x1 - x0 * x0));
  }
  theta = std::min(std::sqrt(chic2 * B) * x, PI);
  return true;
}
inline V3 deflect_by(Rng &g, V3 d, double th) {
  double ph = 2 * PI * g.u();
  return unit(to_lab(d, std::sin(th) * std::cos(ph), std::sin(th) * std::sin(ph), std::cos(th)));
}

struct StepResult { int cls; double L; };    // cls: 0 none, 1 boundary, 2 nuclear, 3 range-out

// One condensed-history step (Reading R3 "H1").  Deposits into `tally` (MeV).
// Returns false when the particle is finished.
bool transport_step(opmc_ctx *c, Particle &p, Rng &g, double *tally, Ledger &led, std::vector<Particle> &stack,
                    EventCheck &chk, uint64_t &nsteps, uint64_t &nel, uint64_t &nne, uint64_t &nsec, double *pathlen) {
  const Tables &T = c->T;
  const size_t vox = ((size_t)p.idx[2] * c->ny + p.idx[1]) * c->nx + p.idx[0];
  const int hu = c->hu[vox];
  const Material &m = material_of(c, hu);
  const double rho = density(m, hu), wf = wet_factor(m, rho);
  nsteps++;
  // 1. nuclear distance, face distance, residual range (L69)
  bool nuclear = c->opt_el || c->opt_ne;
  double Sig = nuclear ? sigma_macro(c, m, rho, p.E, c->opt_el, c->opt_ne, nullptr, nullptr) : 0.0;
  double lam = Sig > 0 ? -std::log(g.u()) / Sig : INF;
  int ax, sg; double dface = dist_to_face(c, p.r, p.d, p.idx, ax, sg);
  double R = T.range_gcm2(m.table_id, p.E) / wf;
  double smax = T.s_max > 0 ? T.s_max / wf : INF;
  // 2. step = min (Reading R3.2)
  double dx = lam; int lim = 2;
  if (dface < dx) { dx = dface; lim = 1; }
  if (R < dx) { dx = R; lim = 3; }
  if (smax < dx * (1 - 1e-6)) { dx = smax; lim = 0; }   // s_max binds only when shorter by more than rounding (R3.2)
  // 3-5. random hinge (L69 ref [19]): first leg tau, deflect, second leg
  double e0 = p.E, tau = 0; V3 dnew = p.d;
  if (c->opt_mcs && dx > 0) {
    tau = g.u() * dx;
    p.r = p.r + tau * p.d;
    double th_m;
    if (c->mcs_model == 1 && moliere_angle(c, m, rho, e0, dx, g, th_m)) dnew = deflect_by(g, p.d, th_m);
    else dnew = deflect(g, p.d, highland(T, e0, dx * rho, m.x0));
  }
  double ell = dx - tau; int ax2, sg2; double d2 = dist_to_face(c, p.r, dnew, p.idx, ax2, sg2);
  double L; int cls;
  if (ell >= d2 || lim == 1) {                     // ends on a face: boundary step whatever limited dx; a face-limited
                                                   // step is always carried to the face (L69; Reading R3.5)
    L = tau + d2; p.r = p.r + d2 * dnew;
    double face = sg2 > 0 ? (p.idx[ax2] + 1) * c->d[ax2] : p.idx[ax2] * c->d[ax2];
    (ax2 == 0 ? p.r.x : ax2 == 1 ? p.r.y : p.r.z) = face;
    cls = 1;
  } else { L = dx; p.r = p.r + ell * dnew; cls = lim; }
  p.d = dnew;
  if (pathlen) *pathlen += L;
  // 6. energy loss from the range table (L61-63, Eq.2) + straggling
  double loss, let_mean = 0;
  if (cls == 3) loss = e0;                         // 7. range-out: everything stays here (L71)
  else {
    double r1 = T.range_gcm2(m.table_id, e0) - L * wf;
    double mean = e0 - (r1 > 0 ? T.energy_of_range(m.table_id, r1) : 0.0);
    mean = std::min(std::max(mean, 0.0), e0);
    let_mean = mean;
    loss = c->opt_strag ? straggle(T, g, e0, mean, L * rho, m.zoa) : mean;
  }
  p.E = e0 - loss;
  double dep = loss;
  bool alive = cls != 3;
  if (alive && p.E <= T.e_cut) { dep += p.E; p.E = 0; alive = false; }     // L71 (2)
  #pragma omp atomic
  tally[vox] += dep;
  led.dep += dep;
  score_influence(c, p.spot, vox, dep);
  if (c->score_let && dep > 0 && L > 0) {
    // dose-averaged LET (Reading R9): every proton step weighs its LET, the table's mean energy loss
    // over the step divided by the step length (keV/um = 0.1 MeV/cm; a proton that ranges out: its energy over its
    // residual range), with the energy the step deposits; heavy recoils and fragments do not enter (L282)
    const double mean_step = cls == 3 ? e0 : let_mean;
    const double let_kev_um = 0.1 * mean_step / L;
    #pragma omp atomic
    c->let_num[vox] += dep * let_kev_um;
    #pragma omp atomic
    c->let_den[vox] += dep;
  }
  if (!alive) return false;
  if (cls == 1) {                                                          // boundary: next voxel
    p.idx[ax2] += sg2;
    if (p.idx[ax2] < 0 || p.idx[ax2] >= (ax2 == 0 ? c->nx : ax2 == 1 ? c->ny : c->nz)) { led.esc += p.E; return false; }  // L71 (3)
    return true;
  }
  if (cls != 2) return true;
  // 8. discrete nuclear event at the end point (L71, L75; Reading R5)
  double pel[OPMC_MAX_ELEM], pne[OPMC_MAX_ELEM];
  double tot = sigma_macro(c, m, rho, p.E, c->opt_el, c->opt_ne, pel, pne);
  if (tot <= 0) return true;
  double sel = 0; for (int i = 0; i < T.n_elem; ++i) sel += pel[i];
  bool is_el = g.u() < sel / tot;
  const double *pe = is_el ? pel : pne; double sum = 0; for (int i = 0; i < T.n_elem; ++i) sum += pe[i];
  double u = g.u() * sum; int el = -1;
  for (int i = 0; i < T.n_elem; ++i) if (pe[i] > 0) { el = i; if (u < pe[i]) break; u -= pe[i]; }
  int Z = T.ez[el], A = T.ea[el];
  {
    uint64_t &tally_ev = (is_el ? c->ev_el : c->ev_ne)[el];
    #pragma omp atomic
    tally_ev++;
  }
  auto deposit_here = [&](double e) {
    #pragma omp atomic
    tally[vox] += e;
    led.dep += e;
    score_influence(c, p.spot, vox, e);
  };
  // NB: the event voxel is the START voxel of the step (interior end point => same voxel)
  if (is_el) {
    nel++;
    ElasticOut o = elastic_event(T, Z, A, p.E, g, chk);
    V3 d0 = p.d;
    p.d = unit(to_lab(d0, o.dir_out.x, o.dir_out.y, o.dir_out.z)); p.E = o.T_out;
    if (A == 1) {                                                          // recoil proton is transported (L136)
      if (o.T_rec > T.e_cut) {
        Particle s = p; s.d = unit(to_lab(d0, o.dir_rec.x, o.dir_rec.y, o.dir_rec.z)); s.E = o.T_rec;
        s.pid = g.child_id(0); s.block0 = 0; stack.push_back(s); nsec++;
      } else deposit_here(o.T_rec);
    } else deposit_here(o.T_rec);                                          // recoil nucleus: local (L79 policy)
    if (p.E <= T.e_cut) { deposit_here(p.E); return false; }
    return true;
  }
  nne++;
  std::vector<Sec> secs; Residual Rz;
  double t_in = p.E;
  nonelastic_event(T, c->nuc[el], t_in, g, secs, Rz, chk);
  double ksum = 0, msum = 0; uint32_t kchild = 0;
  for (const Sec &s : secs) {
    ksum += s.ke; msum += T.nmass(s.Z, s.A);
    if (s.Z == 1 && s.A == 1) {                                            // L79: only protons are followed
      if (s.ke > T.e_cut) {
        Particle q = p; q.d = unit(to_lab(p.d, s.dir.x, s.dir.y, s.dir.z)); q.E = s.ke;
        q.pid = g.child_id(kchild++); q.block0 = 0; stack.push_back(q); nsec++;
      } else deposit_here(s.ke);
    } else if (s.Z == 0) led.neu += s.ke;                                  // neutrons: not transported
    else deposit_here(s.ke);                                               // d,t,3He,alpha: local
  }
  double Mres = Rz.mass_gs + Rz.estar, kres = std::sqrt(dot(Rz.P, Rz.P) + Mres * Mres) - Mres;
  if (Rz.A == 1 && Rz.Z == 0) led.neu += kres; else deposit_here(kres);
  led.gam += Rz.estar;                                                     // L79: no photon evaporation
  led.q += msum + Rz.mass_gs - MP - T.nmass(Z, A);
  (void)ksum;
  return false;
}

// beam-spot sampler (PAPER.md:L102-106 restated; Reading R2).  false => history never enters the grid.
bool sample_primary(opmc_ctx *c, const opmc_spot *spots, const std::vector<double> &cdf, Rng &g, Particle &p,
                    Ledger &led, double &e0) {
  const Tables &T = c->T;
  double u = g.u(); int s = (int)(std::lower_bound(cdf.begin(), cdf.end(), u) - cdf.begin());
  if (s >= (int)cdf.size()) s = (int)cdf.size() - 1;
  const opmc_spot &sp = spots[s];
  p.spot = s;
  V3 ax = unit(V3{sp.dir[0], sp.dir[1], sp.dir[2]});
  V3 a = std::fabs(ax.z) >= 0.9 ? V3{0, 1, 0} : V3{0, 0, 1};
  V3 ex = unit(cross(a, ax)), ey = cross(ax, ex);
  double u1 = g.u(), u2 = g.u(), rr = std::sqrt(-2 * std::log(u1));
  double g1 = rr * std::cos(2 * PI * u2), g2 = rr * std::sin(2 * PI * u2);
  V3 r = V3{sp.pos_cm[0] - c->org[0], sp.pos_cm[1] - c->org[1], sp.pos_cm[2] - c->org[2]} + (sp.sigma_x_cm * g1) * ex + (sp.sigma_y_cm * g2) * ey;
  V3 d = ax;
  if (sp.div_x_rad > 0 || sp.div_y_rad > 0) {
    double u3 = g.u(), u4 = g.u(), r2 = std::sqrt(-2 * std::log(u3));
    d = unit(ax + (sp.div_x_rad * r2 * std::cos(2 * PI * u4)) * ex + (sp.div_y_rad * r2 * std::sin(2 * PI * u4)) * ey);
  }
  double E = sp.e_mev;
  if (sp.sigma_e_mev > 0) E += sp.sigma_e_mev * g.gauss();
  E = std::max(E, 0.0);
  e0 = E;
  const double size[3] = {c->nx * c->d[0], c->ny * c->d[1], c->nz * c->d[2]};
  auto ray_box = [&](V3 o, V3 dd, double &tin) {      // entry distance (>= 0) or miss
    double t0 = 0, t1 = INF; const double oo[3] = {o.x, o.y, o.z}, dv[3] = {dd.x, dd.y, dd.z};
    for (int k = 0; k < 3; ++k) {
      if (dv[k] == 0) { if (oo[k] < 0 || oo[k] > size[k]) return false; continue; }
      double ta = (0 - oo[k]) / dv[k], tb = (size[k] - oo[k]) / dv[k];
      if (ta > tb) std::swap(ta, tb);
      t0 = std::max(t0, ta); t1 = std::min(t1, tb);
    }
    tin = t0; return t0 < t1;
  };
  double tin;
  if (!ray_box(r, d, tin)) { led.esc += E; return false; }
  if (tin > 0) {
    // single air step to the CT edge (L106): hinge, Highland, mean loss + straggling; nuclear omitted (R2)
    const Material &air = material_of(c, -1000);
    double rho = density(air, -1000), wf = wet_factor(air, rho);
    double tau = g.u() * tin;
    V3 rh = r + tau * d, dn = d;
    if (c->opt_mcs) dn = deflect(g, d, highland(T, E, tin * rho, air.x0));
    double t2;
    if (!ray_box(rh, dn, t2)) { led.esc += E; return false; }
    double L = tau + t2; r = rh + t2 * dn; d = dn;
    double r1 = T.range_gcm2(air.table_id, E) - L * wf;
    double mean = std::min(std::max(E - (r1 > 0 ? T.energy_of_range(air.table_id, r1) : 0.0), 0.0), E);
    double loss = c->opt_strag ? straggle(T, g, E, mean, L * rho, air.zoa) : mean;
    led.air += loss; E -= loss;
    if (E <= T.e_cut) { led.air += E; return false; }
  }
  double rv[3] = {r.x, r.y, r.z}; const double dv[3] = {d.x, d.y, d.z}; const int nn[3] = {c->nx, c->ny, c->nz};
  for (int k = 0; k < 3; ++k) {
    rv[k] = std::min(std::max(rv[k], 0.0), size[k]);
    int i = (int)std::floor(rv[k] / c->d[k]);
    if (i * c->d[k] == rv[k] && dv[k] < 0) i -= 1;
    p.idx[k] = std::min(std::max(i, 0), nn[k] - 1);
  }
  p.r = {rv[0], rv[1], rv[2]}; p.d = d; p.E = E; p.pid = 0; p.block0 = 0;
  return true;
}

void run_history(opmc_ctx *c, const opmc_spot *spots, const std::vector<double> &cdf, uint64_t seed, uint64_t h,
                 double *tally, opmc_counters &cn, EventCheck &chk, int max_steps, double *state_out) {
  Ledger led; double e0 = 0;
  std::vector<Particle> stack;
  Rng g0(seed, h, 0);
  Particle p0;
  bool ok = sample_primary(c, spots, cdf, g0, p0, led, e0);
  cn.e_source += e0;
  if (!ok) cn.n_missed++;
  uint64_t nsteps = 0, nel = 0, nne = 0, nsec = 0; double pathlen = 0;
  bool first = true;
  if (ok) stack.push_back(p0);
  while (!stack.empty()) {
    Particle p = stack.back(); stack.pop_back();
    Rng gl(seed, h, p.pid, p.block0);
    Rng &g = first ? g0 : gl;                      // the primary continues the stream used by the sampler
    int steps = 0;
    while (transport_step(c, p, g, tally, led, stack, chk, nsteps, nel, nne, nsec, first ? &pathlen : nullptr)) {
      if (max_steps > 0 && ++steps >= max_steps) break;
    }
    if (first && state_out) {
      double o[8] = {p.r.x, p.r.y, p.r.z, p.d.x, p.d.y, p.d.z, p.E, pathlen};
      std::memcpy(state_out, o, sizeof(o));
    }
    cn.n_draws += first ? 0 : gl.ndraws;
    first = false;
    if (max_steps > 0) break;
  }
  cn.n_draws += g0.ndraws;
  cn.n_steps += nsteps; cn.n_elastic += nel; cn.n_nonelastic += nne; cn.n_secondary_protons += nsec;
  cn.e_deposit += led.dep; cn.e_escape += led.esc; cn.e_neutron += led.neu; cn.e_gamma += led.gam; cn.e_q += led.q; cn.e_air += led.air;
  if (max_steps <= 0) {
    double resid = std::fabs(e0 - (led.dep + led.esc + led.neu + led.gam + led.q + led.air));
    cn.max_ledger_residual = std::max(cn.max_ledger_residual, resid);
  }
}

void merge(opmc_counters &a, const opmc_counters &b, const EventCheck &chk) {
  a.n_steps += b.n_steps; a.n_draws += b.n_draws; a.n_elastic += b.n_elastic; a.n_nonelastic += b.n_nonelastic;
  a.n_secondary_protons += b.n_secondary_protons; a.n_missed += b.n_missed; a.n_inc_tries += chk.inc_tries;
  a.e_source += b.e_source; a.e_deposit += b.e_deposit; a.e_escape += b.e_escape; a.e_neutron += b.e_neutron;
  a.e_gamma += b.e_gamma; a.e_q += b.e_q; a.e_air += b.e_air;
  a.max_ledger_residual = std::max(a.max_ledger_residual, b.max_ledger_residual);
  a.max_event_residual = std::max(a.max_event_residual, chk.max_resid);
  a.n_zab_violations += chk.zab_bad;
  a.n_inc_guard_trips += chk.guard_trips; a.n_inc_stack_trips += chk.stack_trips;
  a.inc_max_stack = std::max(a.inc_max_stack, chk.max_stack); a.inc_max_out = std::max(a.inc_max_out, chk.max_out);
}

int fail(opmc_ctx *c, const char *msg) { if (c) c->err = msg; return -1; }
std::vector<double> spot_cdf(const opmc_spot *s, int n) {
  std::vector<double> cdf(n); double tot = 0;
  for (int i = 0; i < n; ++i) tot += s[i].weight;
  double acc = 0; for (int i = 0; i < n; ++i) { acc += s[i].weight; cdf[i] = acc / tot; }
  cdf[n - 1] = 1.0;
  return cdf;
}
}  // namespace

extern "C" {

int opmc_create(opmc_ctx **out) { if (!out) return -1; *out = new opmc_ctx(); return 0; }
void opmc_destroy(opmc_ctx *c) { delete c; }
const char *opmc_last_error(opmc_ctx *c) { return c ? c->err.c_str() : "null context"; }

int opmc_load_physics_tables(opmc_ctx *c, const opmc_tables *t) {
  if (!c || !t) return fail(c, "null argument");
  if (t->n_e < 4 || t->n_r < 4 || t->n_sr < 1 || t->n_elem < 1 || t->n_elem > OPMC_MAX_ELEM) return fail(c, "bad table sizes");
  Tables &T = c->T;
  T.n_e = t->n_e; T.n_sr = t->n_sr; T.n_r = t->n_r; T.n_elem = t->n_elem; T.zdim = t->mass_zdim; T.adim = t->mass_adim;
  T.e_min = t->e_min; T.e_max = t->e_max; T.dlne = (std::log(T.e_max) - std::log(T.e_min)) / (T.n_e - 1);
  auto cp = [](std::vector<double> &v, const double *p, size_t n) { v.assign(p, p + n); };
  cp(T.stop, t->stop_mass, (size_t)T.n_sr * T.n_e); cp(T.lnR, t->ln_range, (size_t)T.n_sr * T.n_e);
  cp(T.lnR2, t->ln_range_d2, (size_t)T.n_sr * T.n_e); cp(T.lnRlo, t->ln_r_lo, T.n_sr); cp(T.lnRhi, t->ln_r_hi, T.n_sr);
  cp(T.lnE, t->ln_energy, (size_t)T.n_sr * T.n_r); cp(T.lnE2, t->ln_energy_d2, (size_t)T.n_sr * T.n_r);
  cp(T.sne, t->sigma_ne_mb, (size_t)T.n_elem * T.n_e); cp(T.sel, t->sigma_el_mb, (size_t)T.n_elem * T.n_e);
  cp(T.mass, t->nuclear_mass, (size_t)T.zdim * T.adim); cp(T.ek, t->evap_k, (size_t)6 * T.zdim); cp(T.ec, t->evap_c, (size_t)6 * T.zdim);
  T.ez.assign(t->elem_z, t->elem_z + T.n_elem); T.ea.assign(t->elem_a, t->elem_a + T.n_elem);
  for (int s = 0; s < T.n_sr; ++s) for (int i = 1; i < T.n_e; ++i)
    if (!(T.lnR[s * T.n_e + i] > T.lnR[s * T.n_e + i - 1])) return fail(c, "range table not monotone");
  if (t->mol_n > 1 && t->mol_c0 && t->mol_c1 && t->mol_c2) {
    T.mol_c0.assign(t->mol_c0, t->mol_c0 + t->mol_n); T.mol_c1.assign(t->mol_c1, t->mol_c1 + t->mol_n); T.mol_c2.assign(t->mol_c2, t->mol_c2 + t->mol_n);
    T.mol_dth = t->mol_dtheta;
  }
  T.e_cut = t->e_cut; T.highland = t->highland_factor; T.kappa_g = t->kappa_gauss; T.s_max = t->s_max_wet_cm; T.n_batches = t->n_batches;
  c->nuc.assign(T.n_elem, Nucleus());
  for (int i = 0; i < T.n_elem; ++i) if (T.ea[i] > 1) {
    if (T.nmass(T.ez[i], T.ea[i]) <= 0) return fail(c, "element missing from mass table");
    c->nuc[i] = build_nucleus(T, T.ez[i], T.ea[i]);
    c->nuc[i].step_guard = c->inc_step_guard;
  }
  T.loaded = true;
  return 0;
}

int opmc_set_hu_materials(opmc_ctx *c, const opmc_hu_bin *b, int n) {
  if (!c || !b || n < 1) return fail(c, "null/empty materials");
  if (!c->T.loaded) return fail(c, "load physics tables first");
  c->mats.clear();
  for (int i = 0; i < n; ++i) {
    if (b[i].hu_hi <= b[i].hu_lo || (i > 0 && b[i].hu_lo != b[i - 1].hu_hi)) return fail(c, "bins must be sorted and contiguous");
    double sw = 0; for (int k = 0; k < OPMC_MAX_ELEM; ++k) sw += b[i].w[k];
    if (std::fabs(sw - 1) > 1e-6) return fail(c, "mass fractions must sum to 1");
    if (b[i].table_id < 0 || b[i].table_id >= c->T.n_sr) return fail(c, "bad table id");
    Material m; m.hu_lo = b[i].hu_lo; m.hu_hi = b[i].hu_hi; m.rho_lo = b[i].rho_lo; m.rho_hi = b[i].rho_hi;
    std::memcpy(m.w, b[i].w, sizeof(m.w)); m.f_m = b[i].f_m; m.x0 = b[i].x0_gcm2; m.table_id = b[i].table_id;
    m.zoa = 0; for (int k = 0; k < c->T.n_elem; ++k) m.zoa += m.w[k] * c->T.ez[k] / c->T.ea[k];
    c->mats.push_back(m);
  }
  return 0;
}

int opmc_load_ct(opmc_ctx *c, const int16_t *hu, int nx, int ny, int nz, double dx, double dy, double dz, const double origin[3]) {
  if (!c || !hu) return fail(c, "null argument");
  if (nx < 1 || ny < 1 || nz < 1 || !(dx > 0) || !(dy > 0) || !(dz > 0) || (double)nx * ny * nz >= 2147483648.0) return fail(c, "bad grid");
  c->nx = nx; c->ny = ny; c->nz = nz; c->d[0] = dx; c->d[1] = dy; c->d[2] = dz;
  for (int k = 0; k < 3; ++k) c->org[k] = origin ? origin[k] : 0.0;
  c->hu.assign(hu, hu + (size_t)nx * ny * nz);
  c->roi_vox.clear(); c->roi_map.clear(); c->dij.clear();
  return 0;
}

int opmc_set_option(opmc_ctx *c, const char *key, double v) {
  if (!c || !key) return -1;
  std::string k(key);
  if (k == "straggling") c->opt_strag = v != 0; else if (k == "mcs") c->opt_mcs = v != 0;
  else if (k == "elastic") c->opt_el = v != 0; else if (k == "nonelastic") c->opt_ne = v != 0;
  else if (k == "s_max_wet_cm") c->T.s_max = v; else if (k == "n_batches") c->T.n_batches = (int)v;
  else if (k == "threads") c->threads = (int)v; else if (k == "score_letd") c->score_let = v != 0;
  else if (k == "inc_step_guard") { if (v < 1) return fail(c, "inc_step_guard must be >= 1"); c->inc_step_guard = (long)v; for (Nucleus &n : c->nuc) n.step_guard = c->inc_step_guard; }
  else if (k == "mcs_model") { if ((v != 0 && v != 1) || (v == 1 && c->T.mol_c0.empty())) return fail(c, "mcs_model: 0 or 1 (1 needs the Moliere tables)"); c->mcs_model = (int)v; }
  else return fail(c, "unknown option");
  return 0;
}

int opmc_simulate(opmc_ctx *c, const opmc_spot *spots, int nspots, uint64_t n, uint64_t seed, double *dose, double *sigma) {
  if (!c || !spots || nspots < 1 || !dose || !sigma) return fail(c, "null argument");
  if (!c->T.loaded || c->mats.empty() || c->hu.empty()) return fail(c, "call order: tables, materials, ct, simulate");
  const size_t nv = c->hu.size(); const int B = c->T.n_batches;
  if (B < 2) return fail(c, "need >= 2 batches");
  if (n < (uint64_t)B) return fail(c, "n_histories must be at least n_batches");   // groups of N/10 histories
  std::vector<double> cdf = spot_cdf(spots, nspots), tally(nv), s1(nv, 0.0), s2(nv, 0.0);
  c->cnt = opmc_counters{};
  for (int i = 0; i < OPMC_MAX_ELEM; ++i) { c->ev_el[i] = 0; c->ev_ne[i] = 0; }
  if (c->score_let) { c->let_num.assign(nv, 0.0); c->let_den.assign(nv, 0.0); }
  c->dij_spots = nspots;
  if (!c->roi_map.empty()) c->dij.assign((size_t)nspots * c->roi_vox.size(), 0.0);
#ifdef _OPENMP
  if (c->threads > 0) omp_set_num_threads(c->threads);
#endif
  for (int b = 0; b < B; ++b) {                      // PAPER.md:L134 "10 groups of N/10"
    // batch of history h is floor(h*B/N): contiguous ranges
    uint64_t h0 = (uint64_t)(((__uint128_t)b * n + B - 1) / B), h1 = (uint64_t)(((__uint128_t)(b + 1) * n + B - 1) / B);
    std::fill(tally.begin(), tally.end(), 0.0);
    #pragma omp parallel
    {
      opmc_counters cn{}; EventCheck chk;
      #pragma omp for schedule(dynamic, 64)
      for (int64_t h = (int64_t)h0; h < (int64_t)h1; ++h) run_history(c, spots, cdf, seed, (uint64_t)h, tally.data(), cn, chk, 0, nullptr);
      #pragma omp critical
      merge(c->cnt, cn, chk);
    }
    double nb = (double)(h1 - h0);
    for (size_t v = 0; v < nv; ++v) {
      if (tally[v] == 0 || nb == 0) continue;
      int hu = c->hu[v]; const Material &m = material_of(c, hu);
      double mass_g = density(m, hu) * c->d[0] * c->d[1] * c->d[2];
      double db = tally[v] / mass_g / nb * MEV_PER_G_TO_GY;              // Gy per primary (Reading R8)
      s1[v] += db; s2[v] += db * db;
    }
  }
  // influence matrix: MeV -> Gy per primary history of the call (rows then add up to the dose when B divides n)
  for (size_t i = 0; !c->roi_map.empty() && i < (size_t)nspots; ++i)
    for (size_t j = 0; j < c->roi_vox.size(); ++j) {
      int hu = c->hu[c->roi_vox[j]]; const Material &m = material_of(c, hu);
      c->dij[i * c->roi_vox.size() + j] *= MEV_PER_G_TO_GY / (density(m, hu) * c->d[0] * c->d[1] * c->d[2] * (double)n);
    }
  for (size_t v = 0; v < nv; ++v) {                  // PAPER.md:L138 "total and RMS dose" (Reading R8)
    double mean = s1[v] / B, var = (s2[v] - B * mean * mean) / ((double)B * (B - 1));
    dose[v] = mean; sigma[v] = var > 0 ? std::sqrt(var) : 0.0;
  }
  return 0;
}

int opmc_nonelastic(opmc_ctx *c, int Z, int A, double e, uint64_t n, uint64_t seed, opmc_secondary *out, uint64_t cap,
                    uint32_t *off, uint64_t *n_out) {
  if (!c || !off || !n_out || (!out && cap > 0)) return fail(c, "null argument");
  if (!c->T.loaded) return fail(c, "load physics tables first");
  if (A < 2 || c->T.nmass(Z, A) <= 0 || c->T.nmass(Z - 1, A - 1) <= 0 || c->T.nmass(Z, A - 1) <= 0) return fail(c, "unsupported target");
  Nucleus N = build_nucleus(c->T, Z, A);
  N.step_guard = c->inc_step_guard;
  c->cnt = opmc_counters{};
  EventCheck chk; uint64_t pos = 0; bool overflow = false;
  for (uint64_t ev = 0; ev < n; ++ev) {
    Rng g(seed, ev, 0);
    std::vector<Sec> secs; Residual R;
    nonelastic_event(c->T, N, e, g, secs, R, chk);
    double Mres = R.mass_gs + R.estar;
    secs.push_back({R.Z, R.A, 2, std::sqrt(dot(R.P, R.P) + Mres * Mres) - Mres, norm(R.P) > 0 ? unit(R.P) : V3{0, 0, 1}});
    off[ev] = (uint32_t)pos;
    for (const Sec &s : secs) {
      if (pos < cap) { opmc_secondary o{}; o.Z = (int16_t)s.Z; o.A = (int16_t)s.A; o.origin = (uint8_t)s.origin; o.ke_mev = (float)s.ke;
        o.dir[0] = (float)s.dir.x; o.dir[1] = (float)s.dir.y; o.dir[2] = (float)s.dir.z; out[pos] = o; } else overflow = true;
      pos++;
    }
    c->cnt.e_gamma += R.estar; c->cnt.n_draws += g.ndraws;
  }
  off[n] = (uint32_t)pos; *n_out = pos;
  c->cnt.n_nonelastic = n; c->cnt.n_inc_tries = chk.inc_tries; c->cnt.max_event_residual = chk.max_resid; c->cnt.n_zab_violations = chk.zab_bad;
  c->cnt.n_inc_guard_trips = chk.guard_trips; c->cnt.n_inc_stack_trips = chk.stack_trips; c->cnt.inc_max_stack = chk.max_stack; c->cnt.inc_max_out = chk.max_out;
  if (overflow) return fail(c, "capacity too small"), -3;
  return 0;
}

// Per-spot dose influence ("MC-based IMPT optimisation"; Reading R11): roi_voxels = n_roi linear voxel
// indices (x fastest); the next opmc_simulate calls also fill D[spot][roi] = dose (Gy per primary history of the call)
// that histories of that spot give to that voxel.  n_roi = 0 switches it off.
int opmc_set_dose_influence(opmc_ctx *c, const int32_t *roi_voxels, int n_roi) {
  if (!c || n_roi < 0 || (n_roi > 0 && !roi_voxels)) return fail(c, "bad argument");
  if (c->hu.empty()) return fail(c, "load the CT first");
  c->roi_vox.clear(); c->roi_map.clear(); c->dij.clear();
  if (n_roi == 0) return 0;
  c->roi_map.assign(c->hu.size(), -1);
  for (int j = 0; j < n_roi; ++j) {
    if (roi_voxels[j] < 0 || (size_t)roi_voxels[j] >= c->hu.size() || c->roi_map[roi_voxels[j]] >= 0) { c->roi_map.clear(); return fail(c, "ROI voxel out of range or repeated"); }
    c->roi_map[roi_voxels[j]] = j;
  }
  c->roi_vox.assign(roi_voxels, roi_voxels + n_roi);
  return 0;
}
int opmc_get_dose_influence(opmc_ctx *c, double *out) {
  if (!c || !out) return -1;
  if (c->roi_vox.empty() || c->dij.size() != (size_t)c->dij_spots * c->roi_vox.size() || c->dij.empty()) return fail(c, "no influence matrix: set the ROI and simulate");
  std::memcpy(out, c->dij.data(), c->dij.size() * sizeof(double));
  return 0;
}

// LET_d map of the last opmc_simulate run with "score_letd" on: keV/um, 0 where no proton step deposited energy
int opmc_get_letd(opmc_ctx *c, double *out) {
  if (!c || !out) return -1;
  if (!c->score_let || c->let_num.size() != c->hu.size() || c->let_num.empty()) return fail(c, "no LET_d tally: set score_letd and simulate");
  for (size_t v = 0; v < c->let_num.size(); ++v) out[v] = c->let_den[v] > 0 ? c->let_num[v] / c->let_den[v] : 0.0;
  return 0;
}
int opmc_get_counters(opmc_ctx *c, opmc_counters *o) { if (!c || !o) return -1; *o = c->cnt; return 0; }

// ---------------------------------------------------------------- test hooks
void opmc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) { philox(ctr, key, out); }
double opmc_test_range_gcm2(opmc_ctx *c, int t, double e) { return c->T.range_gcm2(t, e); }
double opmc_test_energy_of_range(opmc_ctx *c, int t, double r) { return c->T.energy_of_range(t, r); }
int opmc_test_straggle(opmc_ctx *c, double e, double mean, double rhoL, double zoa, uint64_t n, uint64_t seed, double *out) {
  for (uint64_t i = 0; i < n; ++i) { Rng g(seed, i, 0); out[i] = straggle(c->T, g, e, mean, rhoL, zoa); }
  return 0;
}
int opmc_test_first_steps(opmc_ctx *c, const opmc_spot *spot, uint64_t n, uint64_t seed, int max_steps, double *out) {
  std::vector<double> cdf = spot_cdf(spot, 1), tally(c->hu.size(), 0.0);
  opmc_counters cn{}; EventCheck chk;
  for (uint64_t h = 0; h < n; ++h) run_history(c, spot, cdf, seed, h, tally.data(), cn, chk, max_steps, out + 8 * h);
  return 0;
}
int opmc_test_elastic(opmc_ctx *c, int Z, int A, double t, uint64_t n, uint64_t seed, double *out) {
  EventCheck chk;
  for (uint64_t i = 0; i < n; ++i) {
    Rng g(seed, i, 0); ElasticOut o = elastic_event(c->T, Z, A, t, g, chk);
    out[4 * i] = o.t_gev2; out[4 * i + 1] = o.T_out; out[4 * i + 2] = o.T_rec;
    out[4 * i + 3] = std::acos(std::min(1.0, std::max(-1.0, dot(o.dir_out, o.dir_rec))));
  }
  c->cnt.max_event_residual = chk.max_resid;
  return 0;
}
double opmc_test_inc_uniform_sphere(double radius, double rho, double sigma_mb, double t, uint64_t n, uint64_t seed) {
  Tables T; T.zdim = 2; T.adim = 2; T.mass = {0, MN, 0, MP};
  Nucleus N; N.Z = 0; N.A = 1; N.nshell = 1; N.rmax = radius; N.rout[0] = radius; N.pauli = false; N.const_sigma_mb = sigma_mb;
  for (int ty = 0; ty < 2; ++ty) { N.rho[ty][0] = ty == 1 ? rho : 0.0; N.pF[ty][0] = 0; N.EF[ty][0] = 0; N.V[ty][0] = 0; }
  N.coulomb = -1e9;                                        // nothing is ever trapped
  uint64_t hits = 0;
  for (uint64_t i = 0; i < n; ++i) {
    Rng g(seed, i, 0); std::vector<Sec> o; Residual R;
    // count collisions through the attempt's return path: an attempt with >= 1 collision either succeeds or
    // fails only on the residual bookkeeping (irrelevant here), so re-derive from the number of outgoing nucleons
    inc_attempt(T, N, t, g, o, R);
    if (o.size() >= 2) hits++;                             // Pauli off, no trapping: each collision adds a nucleon
  }
  return (double)hits / (double)n;
}
double opmc_test_nucleus(opmc_ctx *c, int Z, int A, double *out) {
  Nucleus N = build_nucleus(c->T, Z, A);
  for (int k = 0; k < 15; ++k) { double *o = out + 6 * k; o[0] = N.rout[k]; o[1] = N.rho[0][k]; o[2] = N.rho[1][k]; o[3] = N.pF[0][k]; o[4] = N.EF[0][k]; o[5] = N.V[0][k]; }
  return N.rmax;
}
// the neutron side of the same model (test hook, no arithmetic of its own): out[15][3] = pF_n, EF_n, V_n
double opmc_test_nucleus_neutron(opmc_ctx *c, int Z, int A, double *out) {
  Nucleus N = build_nucleus(c->T, Z, A);
  for (int k = 0; k < 15; ++k) { double *o = out + 3 * k; o[0] = N.pF[1][k]; o[1] = N.EF[1][k]; o[2] = N.V[1][k]; }
  return N.coulomb;
}
double opmc_test_fermi_p2(opmc_ctx *c, int Z, int A, uint64_t n, uint64_t seed) {
  Nucleus N = build_nucleus(c->T, Z, A); double acc = 0;
  Rng g(seed, 0, 0);
  for (uint64_t i = 0; i < n; ++i) { double q = N.pF[0][0] * std::cbrt(g.u()); V3 v = q * isotropic(g); acc += dot(v, v); }
  return acc / n / (N.pF[0][0] * N.pF[0][0]);
}
int opmc_test_evap_first(opmc_ctx *c, int Z, int A, double estar, uint32_t mask, uint64_t n, uint64_t seed, double *widths,
                         int32_t *och, double *oeps, double *ocos) {
  Channel ch[6]; evap_channels(c->T, Z, A, estar, 0x3F, ch);
  for (int j = 0; j < 6; ++j) widths[j] = ch[j].open ? ch[j].width : 0.0;
  for (uint64_t i = 0; i < n; ++i) {
    Rng g(seed, i, 0); Residual R{Z, A, estar, V3{0, 0, 0}, c->T.nmass(Z, A)}; Sec s; double e = 0, cs = 0;
    och[i] = evap_emit(c->T, R, g, mask, s, &e, &cs); oeps[i] = e; ocos[i] = cs;
  }
  return 0;
}
// n samples of cos(theta_cm) of NN elastic scattering at lab momentum p_lab (GeV/c) and CM momentum pcm (MeV/c)
int opmc_test_nn_cos(int same_type, double p_lab_gev, double pcm_mev, uint64_t n, uint64_t seed, double *out) {
  for (uint64_t i = 0; i < n; ++i) { Rng g(seed, i, 0); out[i] = sample_nn_cos(g, same_type != 0, p_lab_gev, pcm_mev); }
  return 0;
}
// Cascade attempts on a hand-made nucleus of ns concentric shells (outer radii rout[ns]; per nucleon type t = 0 proton,
// 1 neutron: density rho[t*ns+k], Fermi momentum pF[t*ns+k], potential depth V[t*ns+k]); incident proton of kinetic
// energy t_in.  Attempt i uses the stream (seed, i).  out_n[i] = number of nucleons that left the nucleus, or -1 - that
// number when the attempt was rejected; out_rec[i][4][5] = type, kinetic energy, direction of the first four of them.
int opmc_test_inc_custom(int ns, const double *rout, const double *rho, const double *pF, const double *V, double coulomb,
                         int pauli, double const_sigma_mb, double t_in, uint64_t n, uint64_t seed, int32_t *out_n,
                         double *out_rec) {
  if (ns < 1 || ns > NSHELL_MAX) return -1;
  Tables T; T.zdim = 2; T.adim = 2; T.mass = {0, MN, 0, MP};
  Nucleus N; N.Z = 0; N.A = 1; N.nshell = ns; N.rmax = rout[ns - 1]; N.pauli = pauli != 0; N.const_sigma_mb = const_sigma_mb;
  N.coulomb = coulomb;
  for (int t = 0; t < 2; ++t) for (int k = 0; k < ns; ++k) {
    const double m = nucleon_mass(t);
    N.rout[k] = rout[k]; N.rho[t][k] = rho[t * ns + k]; N.pF[t][k] = pF[t * ns + k]; N.V[t][k] = V[t * ns + k];
    N.EF[t][k] = std::sqrt(N.pF[t][k] * N.pF[t][k] + m * m) - m;
  }
  for (uint64_t i = 0; i < n; ++i) {
    Rng g(seed, i, 0); std::vector<Sec> o; Residual R;
    const bool ok = inc_attempt(T, N, t_in, g, o, R);
    out_n[i] = ok ? (int32_t)o.size() : -1 - (int32_t)o.size();
    for (size_t k = 0; k < 4; ++k) {
      double *r = out_rec + (i * 4 + k) * 5;
      if (k < o.size()) { r[0] = o[k].Z == 1 ? 0 : 1; r[1] = o[k].ke; r[2] = o[k].dir.x; r[3] = o[k].dir.y; r[4] = o[k].dir.z; }
      else { r[0] = -1; r[1] = r[2] = r[3] = r[4] = 0; }
    }
  }
  return 0;
}
// n primaries of a multi-spot plan straight from the beam-spot sampler: out[n][8] = spot index, x, y, z (grid frame, at
// the grid entry), u, v, w, E; spot index -1 = the history never enters the grid
int opmc_test_sample_primaries(opmc_ctx *c, const opmc_spot *spots, int nspots, uint64_t n, uint64_t seed, double *out) {
  if (!c || !spots || nspots < 1 || c->hu.empty()) return -1;
  std::vector<double> cdf = spot_cdf(spots, nspots);
  for (uint64_t h = 0; h < n; ++h) {
    Rng g(seed, h, 0); Particle p; Ledger led; double e0 = 0;
    const bool ok = sample_primary(c, spots, cdf, g, p, led, e0);
    double *o = out + 8 * h;
    o[0] = ok ? p.spot : -1; o[1] = p.r.x; o[2] = p.r.y; o[3] = p.r.z; o[4] = p.d.x; o[5] = p.d.y; o[6] = p.d.z; o[7] = ok ? p.E : e0;
  }
  return 0;
}
// events of the last opmc_simulate per class and target element: out[0..7] elastic, out[8..15] non-elastic
int opmc_test_event_counts(opmc_ctx *c, uint64_t *out) {
  if (!c || !out) return -1;
  for (int i = 0; i < OPMC_MAX_ELEM; ++i) { out[i] = c->ev_el[i]; out[OPMC_MAX_ELEM + i] = c->ev_ne[i]; }
  return 0;
}
double opmc_test_cugnon(int which, double p) {
  switch (which) { case 0: return cug_sigma_pp(p); case 1: return cug_sigma_np(p); case 2: return cug_b_pp(p); case 3: return cug_b_np(p); default: return cug_a_np(p); }
}
}  // extern "C"
