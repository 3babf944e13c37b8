// pmc_api.cu — libpmc: context, host-side table preparation, the event-based transport scheduler and the C-ABI
// of include/pmc.h.  No torch types, no CPU fallback: every step of the path runs in the kernels of
// pmc_transport.cuh / pmc_nuclear.cuh.
#include "../../include/pmc.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <algorithm>
#include <string>
#include <vector>

#include "pmc_device.cuh"
#include "pmc_transport.cuh"
#include "pmc_nuclear.cuh"
#include "pmc_gamma.cuh"

using namespace pmc;

namespace {

constexpr double NAVO = 6.02214076e23;
constexpr double PI_D = 3.14159265358979323846;

struct HostMat { pmc_hu_bin b; double zoa; };

// Device scratch comes from the context's allocator: cudaMalloc / cudaFree by default, or the pair of callbacks given to
// pmc_create_with_allocator (so that e.g. PyTorch's caching allocator owns the queues and tallies).
struct Allocator { pmc_alloc_fn alloc = nullptr; pmc_free_fn free = nullptr; void *user = nullptr; };
struct DevBufBase {
  const Allocator *A = nullptr;
  virtual void release() = 0;
  virtual ~DevBufBase() {}
};
// every DevBuf constructed while this points to a list (i.e. while a pmc_ctx is being constructed) is entered into it
thread_local std::vector<DevBufBase *> *tl_registry = nullptr;

template <typename T>
struct DevBuf : DevBufBase {
  T *p = nullptr; size_t n = 0;
  DevBuf() { if (tl_registry) tl_registry->push_back(this); }
  cudaError_t alloc(size_t count) {
    if (count <= n && p) return cudaSuccess;
    release();
    cudaError_t e = cudaSuccess;
    if (A && A->alloc) { p = static_cast<T *>(A->alloc(count * sizeof(T), A->user)); if (!p) e = cudaErrorMemoryAllocation; }
    else e = cudaMalloc(&p, count * sizeof(T));
    if (e == cudaSuccess) n = count; else p = nullptr;
    return e;
  }
  cudaError_t upload(const std::vector<T> &h, cudaStream_t s) {
    cudaError_t e = alloc(h.size() ? h.size() : 1);
    if (e != cudaSuccess) return e;
    if (h.empty()) return cudaSuccess;
    return cudaMemcpyAsync(p, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice, s);
  }
  void release() override {
    if (p) { if (A && A->free) A->free(p, A->user); else cudaFree(p); }
    p = nullptr; n = 0;
  }
};

struct QueueMem {
  DevBuf<float> f; DevBuf<int> vox; DevBuf<uint32_t> u; DevBuf<uint32_t> count;
  Queue q{};
  cudaError_t alloc(uint32_t cap) {
    cudaError_t e;
    if ((e = f.alloc((size_t)cap * 7)) != cudaSuccess) return e;
    if ((e = vox.alloc(cap)) != cudaSuccess) return e;
    if ((e = u.alloc((size_t)cap * 4)) != cudaSuccess) return e;
    if ((e = count.alloc(1)) != cudaSuccess) return e;
    q.x = f.p; q.y = f.p + cap; q.z = f.p + 2ull * cap; q.u = f.p + 3ull * cap; q.v = f.p + 4ull * cap; q.w = f.p + 5ull * cap;
    q.e = f.p + 6ull * cap; q.vox = vox.p; q.hist = u.p; q.pid = u.p + cap; q.blk = u.p + 2ull * cap; q.aux = u.p + 3ull * cap;
    q.count = count.p; q.cap = cap;
    return cudaSuccess;
  }
};

}  // namespace

struct pmc_ctx {
  Allocator allocator; std::vector<DevBufBase *> bufs;   // every device buffer of the context (filled by pmc_create)
  int device = 0; cudaStream_t stream = nullptr;
  std::string err;
  // host copies
  bool have_tables = false, have_mats = false, have_ct = false, tables_dirty = true;
  int n_e = 0, n_r = 0, n_sr = 0, n_elem = 0, zdim = 0, adim = 0;
  double e_min = 0, e_max = 0;
  std::vector<double> h_lnR, h_lnR2, h_lnrlo, h_lnrhi, h_lnE, h_lnE2, h_sne, h_sel, h_mass, h_ek, h_ec;
  std::vector<int> ez, ea;
  std::vector<float> h_mol; int mol_n = 0; double mol_dth = 0; int mcs_model = 0; DevBuf<float> d_mol;
  double e_cut = 0.1, highland = 1.07, kappa_g = 10, s_max = 0.2; int n_batches = 10;
  bool opt_strag = true, opt_mcs = true, opt_el = true, opt_ne = true; int aggregate = 0; bool profile = true, skip_tally = false;
  uint64_t chunk = 1u << 24, history_offset = 0;
  std::vector<HostMat> mats;
  // device tables
  DevBuf<float> d_lnR, d_lnR2, d_lnE, d_lnE2, d_sel, d_sne, d_sigbin, d_ek, d_ec;
  DevBuf<double> d_mass; DevBuf<MatBin> d_bins; DevBuf<uint8_t> d_lut; DevBuf<int2> d_lut2; DevBuf<Nucleus> d_nuc, d_nuc1;
  std::vector<Nucleus> h_nuc;
  Tables T{}; Grid G{}; double origin[3] = {0, 0, 0};
  DevBuf<int16_t> d_hu_own;
  // scratch
  QueueMem qa, qb, qev, qel, qne, qres; DevBuf<uint32_t> d_resza; DevBuf<float> d_resp;
  DevBuf<uint32_t> d_head; DevBuf<Counters> d_cnt; DevBuf<float> d_tally, d_out, d_let;
  bool score_let = false, have_let = false;
  DevBuf<int32_t> d_roimap, d_roivox; uint32_t n_roi = 0; float *dij_dev = nullptr; uint64_t dij_cap = 0;
  DevBuf<SpotDev> d_spots; DevBuf<double> d_cdf; DevBuf<uint32_t> d_guide;
  DevBuf<SecRec> d_slots; DevBuf<uint32_t> d_counts; DevBuf<unsigned long long> d_base; DevBuf<ResRec> d_res;
  DevBuf<GammaOffset> d_goff; DevBuf<unsigned long long> d_gscr;
  uint32_t *h_pinned = nullptr;     // pinned readback word(s)
  uint32_t qcap = 0;
  int n_sm = 148; size_t smem_transport = 0;
  int inc_bpsm = 0, evap_bpsm = 0;     // resident blocks per SM of the two warp-synchronous engines (occupancy API)
  pmc_counters counters{}; pmc_timing timing{};
  cudaEvent_t ev[2] = {nullptr, nullptr};
  std::vector<cudaEvent_t> ev_pool; size_t ev_used = 0; std::vector<float *> ev_acc;
};

namespace {

int fail(pmc_ctx *c, int code, const std::string &msg) { if (c) c->err = msg; return code; }
int cuda_fail(pmc_ctx *c, cudaError_t e, const char *where) {
  return fail(c, PMC_E_CUDA, std::string(where) + ": " + cudaGetErrorString(e));
}
#define CK(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return cuda_fail(c, e__, #call); } while (0)

double h_nmass(const pmc_ctx *c, int z, int a) {
  return (z < 0 || a < 1 || z >= c->zdim || a >= c->adim || z > a) ? 0.0 : c->h_mass[(size_t)z * c->adim + a];
}

// Woods-Saxon density approximated by 15 constant-density shells of a two-component Fermi gas.
// Reading R6.1: c = 1.07 A^(1/3) fm, a = 0.545 fm, r_max at 1 % of the central density, equal radial widths,
// shell density = volume average (Simpson), normalised to A; V = E_F + separation energy; B_C = 1.44 (Z-1)/r_max.
Nucleus build_nucleus(const pmc_ctx *c, int Z, int A) {
  Nucleus n{}; n.Z = Z; n.A = A; n.nshell = NSHELL; n.pauli = 1; n.const_sigma_mb = -1.f;
  const double c0 = 1.07 * std::cbrt((double)A), a = 0.545, rmax = c0 + a * std::log(99.0), dr = rmax / NSHELL;
  double avg[NSHELL], tot = 0;
  auto ws = [&](double r) { return r * r / (1.0 + std::exp((r - c0) / a)); };
  for (int k = 0; k < NSHELL; ++k) {
    const double r0 = k * dr, r1 = (k + 1) * dr; const int M = 256; const double h = (r1 - r0) / M;
    double s = ws(r0) + ws(r1);
    for (int i = 1; i < M; ++i) s += ws(r0 + i * h) * ((i & 1) ? 4.0 : 2.0);
    const double integral = s * h / 3.0, vol = 4 * PI_D / 3 * (r1 * r1 * r1 - r0 * r0 * r0);
    avg[k] = 4 * PI_D * integral / vol; tot += avg[k] * vol; n.rout[k] = (float)r1;
  }
  const double sep[2] = {h_nmass(c, Z - 1, A - 1) + MP_D - h_nmass(c, Z, A), h_nmass(c, Z, A - 1) + MN_D - h_nmass(c, Z, A)};
  for (int k = 0; k < NSHELL; ++k)
    for (int t = 0; t < 2; ++t) {
      const double frac = t == 0 ? (double)Z / A : (double)(A - Z) / A, m = t == 0 ? MP_D : MN_D;
      const double rho = avg[k] * A / tot * frac, pF = 197.3269804 * std::cbrt(3 * PI_D * PI_D * rho);
      const double EF = std::sqrt(pF * pF + m * m) - m;
      n.rho[t][k] = (float)rho; n.pF[t][k] = (float)pF; n.EF[t][k] = (float)EF; n.V[t][k] = (float)(EF + sep[t]);
    }
  n.rmax = (float)rmax; n.coulomb = (float)(1.44 * (Z - 1) / rmax); n.mass = h_nmass(c, Z, A);
  return n;
}

std::vector<float> to_f(const std::vector<double> &v, double scale = 1.0) {
  std::vector<float> o(v.size());
  for (size_t i = 0; i < v.size(); ++i) o[i] = (float)(v[i] * scale);
  return o;
}

// (re)build every device table that depends on tables + materials + options
int sync_tables(pmc_ctx *c) {
  if (!c->tables_dirty) return PMC_OK;
  cudaStream_t s = c->stream;
  Tables &T = c->T;
  T.n_e = c->n_e; T.n_r = c->n_r; T.n_sr = c->n_sr; T.n_elem = c->n_elem; T.zdim = c->zdim; T.adim = c->adim;
  const double dlne = (std::log(c->e_max) - std::log(c->e_min)) / (c->n_e - 1);
  T.ln_emin = (float)std::log(c->e_min); T.ln_emax = (float)std::log(c->e_max); T.inv_dlne = (float)(1.0 / dlne);
  T.e_min = (float)c->e_min; T.e_max = (float)c->e_max;
  T.c_l2 = (float)(std::log(2.0) / dlne); T.c_e0 = (float)(std::log(c->e_min) / dlne);
  T.e_cut = (float)c->e_cut; T.highland = (float)c->highland; T.kappa_g = (float)c->kappa_g; T.s_max = (float)c->s_max;
  T.opt_strag = c->opt_strag; T.opt_mcs = c->opt_mcs; T.opt_el = c->opt_el; T.opt_ne = c->opt_ne;
  CK(c->d_mol.upload(c->h_mol, s)); T.mol_c = c->d_mol.p; T.mol_n = c->mol_n; T.mol_dth = (float)c->mol_dth; T.mcs_model = c->mol_n > 1 ? c->mcs_model : 0;
  CK(c->d_lnR.upload(to_f(c->h_lnR), s)); CK(c->d_lnR2.upload(to_f(c->h_lnR2, dlne * dlne / 6.0), s));
  std::vector<float> e2(c->h_lnE2.size());
  for (int t = 0; t < c->n_sr; ++t) {
    const double h = (c->h_lnrhi[t] - c->h_lnrlo[t]) / (c->n_r - 1);
    T.lnr_lo[t] = (float)c->h_lnrlo[t]; T.lnr_hi[t] = (float)c->h_lnrhi[t]; T.inv_hr[t] = (float)(1.0 / h);
    for (int i = 0; i < c->n_r; ++i) e2[(size_t)t * c->n_r + i] = (float)(c->h_lnE2[(size_t)t * c->n_r + i] * h * h / 6.0);
  }
  CK(c->d_lnE.upload(to_f(c->h_lnE), s)); CK(c->d_lnE2.upload(e2, s));
  CK(c->d_sel.upload(to_f(c->h_sel), s)); CK(c->d_sne.upload(to_f(c->h_sne), s));
  CK(c->d_mass.upload(c->h_mass, s)); CK(c->d_ek.upload(to_f(c->h_ek), s)); CK(c->d_ec.upload(to_f(c->h_ec), s));
  CK(c->d_nuc.upload(c->h_nuc, s));
  T.lnR = c->d_lnR.p; T.lnR2 = c->d_lnR2.p; T.lnE = c->d_lnE.p; T.lnE2 = c->d_lnE2.p; T.sig_el = c->d_sel.p; T.sig_ne = c->d_sne.p;
  T.mass = c->d_mass.p; T.evap_k = c->d_ek.p; T.evap_c = c->d_ec.p; T.nuc = c->d_nuc.p;
  for (int i = 0; i < MAX_ELEM; ++i) { T.elem_z[i] = i < c->n_elem ? c->ez[i] : 0; T.elem_a[i] = i < c->n_elem ? c->ea[i] : 1; }
  T.nbins = (int)c->mats.size();
  if (c->have_mats) {
    const int nb = T.nbins;
    std::vector<MatBin> bins(nb); std::vector<float> sig((size_t)nb * c->n_e);
    for (int b = 0; b < nb; ++b) {
      const pmc_hu_bin &h = c->mats[b].b; MatBin &m = bins[b];
      m.hu_lo = (float)h.hu_lo; m.dhu = (float)((double)h.hu_hi - h.hu_lo); m.inv_dhu = (float)(1.0 / ((double)h.hu_hi - h.hu_lo));
      m.rho_lo = (float)h.rho_lo; m.drho = (float)(h.rho_hi - h.rho_lo); m.slope = (float)((h.rho_hi - h.rho_lo) / ((double)h.hu_hi - h.hu_lo));
      m.lnr_lo = T.lnr_lo[h.table_id]; m.lnr_hi = T.lnr_hi[h.table_id]; m.inv_hr = T.inv_hr[h.table_id];
      m.off_e = 2 * h.table_id * c->n_e; m.off_r = 2 * (c->n_sr * c->n_e + h.table_id * c->n_r);
      m.off_sig = 2 * c->n_sr * (c->n_e + c->n_r) + b * c->n_e;
      m.wet = h.table_id == 0 ? (float)h.f_m : 1.0f; m.inv_x0 = (float)(1.0 / h.x0_gcm2); m.zoa = (float)c->mats[b].zoa; m.table = h.table_id;
      for (int i = 0; i < MAX_ELEM; ++i) m.nfac[i] = i < c->n_elem ? (float)(NAVO * h.w[i] / c->ea[i] * 1e-27) : 0.f;
      double zs = 0; for (int i = 0; i < c->n_elem; ++i) zs += h.w[i] * c->ez[i] * (c->ez[i] + 1.0) / c->ea[i];
      m.zs = (float)zs;
      // macroscopic cross-section per unit density: a sum of tables that are linear in ln E is linear in ln E
      for (int k = 0; k < c->n_e; ++k) {
        double acc = 0;
        for (int i = 0; i < c->n_elem; ++i) {
          const double nf = NAVO * h.w[i] / c->ea[i] * 1e-27;
          if (c->opt_el) acc += nf * c->h_sel[(size_t)i * c->n_e + k];
          if (c->opt_ne) acc += nf * c->h_sne[(size_t)i * c->n_e + k];
        }
        sig[(size_t)b * c->n_e + k] = (float)acc;
      }
    }
    // HU -> bin lookup table over [first bin's upper edge - 1, last bin's lower edge]; HU outside is clamped (L49)
    const int lo = nb > 1 ? c->mats.front().b.hu_hi - 1 : c->mats.front().b.hu_lo;
    const int hi = nb > 1 ? c->mats.back().b.hu_lo : c->mats.front().b.hu_lo;
    std::vector<uint8_t> lut((size_t)(hi - lo + 1));
    for (int hu = lo, b = 0; hu <= hi; ++hu) { while (b < nb - 1 && hu >= c->mats[b].b.hu_hi) ++b; lut[hu - lo] = (uint8_t)b; }
    T.hu_lut_lo = lo; T.hu_lut_n = (int)lut.size();
    // the same table with the density of every HU value beside its bin (step kernel: one 8-byte load instead of the bin's
    // density line); the first and the last bin have one entry each, exact only if their density does not depend on HU
    std::vector<int2> lut2(lut.size());
    for (int hu = lo; hu <= hi; ++hu) {
      const pmc_hu_bin &h = c->mats[lut[hu - lo]].b;
      const int hh = std::min(std::max(hu, h.hu_lo), h.hu_hi);
      const float rho = (float)(h.rho_lo + (h.rho_hi - h.rho_lo) * ((double)hh - h.hu_lo) / ((double)h.hu_hi - h.hu_lo));
      int bits; std::memcpy(&bits, &rho, 4);
      lut2[hu - lo] = make_int2(bits, (int)lut[hu - lo]);
    }
    T.lut_ends_vary = (c->mats.front().b.rho_lo != c->mats.front().b.rho_hi || c->mats.back().b.rho_lo != c->mats.back().b.rho_hi) ? 1 : 0;
    CK(c->d_lut2.upload(lut2, s)); T.hu_lut2 = c->d_lut2.p;
    CK(c->d_bins.upload(bins, s)); CK(c->d_sigbin.upload(sig, s)); CK(c->d_lut.upload(lut, s));
    T.bins = c->d_bins.p; T.sig_bin = c->d_sigbin.p; T.hu_lut = c->d_lut.p;
    c->smem_transport = ((size_t)2 * c->n_sr * c->n_e + (size_t)2 * c->n_sr * c->n_r + (size_t)nb * c->n_e) * 4 + (size_t)nb * sizeof(MatBin) +
                        lut.size() * sizeof(int2) + 32;
    if (c->smem_transport > 200 * 1024) return fail(c, PMC_E_UNSUPPORTED, "tables too large for shared-memory staging");
#define PMC_SMEM_ATTR(M, D, X) CK(cudaFuncSetAttribute(transport_kernel<M, D, X>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem_transport))
    PMC_SMEM_ATTR(0, false, false); PMC_SMEM_ATTR(0, false, true); PMC_SMEM_ATTR(1, false, false); PMC_SMEM_ATTR(1, false, true);
    PMC_SMEM_ATTR(0, true, false); PMC_SMEM_ATTR(1, true, false);
#undef PMC_SMEM_ATTR
  }
  CK(cudaStreamSynchronize(s));
  c->tables_dirty = false;
  return PMC_OK;
}

// one launch instead of six memsets per generation: work-fetch heads and the counts of the queues the generation fills
__global__ void reset_kernel(uint32_t *head4, uint32_t *a, uint32_t *b, uint32_t *c_, uint32_t *d, uint32_t *e) {
  const int t = threadIdx.x;
  if (t < 4) head4[t] = 0u;
  else if (t == 4) *a = 0u; else if (t == 5) *b = 0u; else if (t == 6) *c_ = 0u; else if (t == 7) *d = 0u; else if (t == 8) *e = 0u;
}

// generations enqueued before the host first looks at a queue size, then per look; slots of the per-generation counts
constexpr int GEN_BURST = 6, GEN_MORE = 2, GEN_SLOTS = 64;

int ensure_scratch(pmc_ctx *c, uint64_t chunk) {
  const uint32_t cap = (uint32_t)std::max<uint64_t>(chunk + chunk / 4 + 4096, 8192);
  if (cap > c->qcap) {
    CK(c->qa.alloc(cap)); CK(c->qb.alloc(cap)); CK(c->qev.alloc(cap)); CK(c->qel.alloc(cap)); CK(c->qne.alloc(cap)); CK(c->qres.alloc(cap));
    CK(c->d_resza.alloc(cap)); CK(c->d_resp.alloc((size_t)cap * 3));
    c->qcap = cap;
  }
  CK(c->d_head.alloc(4 + GEN_SLOTS)); CK(c->d_cnt.alloc(1));
  if (!c->h_pinned) CK(cudaMallocHost(&c->h_pinned, 4 * (GEN_SLOTS + 4)));
  if (!c->ev[0]) { CK(cudaEventCreate(&c->ev[0])); CK(cudaEventCreate(&c->ev[1])); }
  if (!c->inc_bpsm) {                  // persistent engines: exactly one wave of blocks
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->inc_bpsm, inc_kernel, 128, 0));
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->evap_bpsm, evap_kernel, 128, 0));
    c->inc_bpsm = std::max(c->inc_bpsm, 1); c->evap_bpsm = std::max(c->evap_bpsm, 1);
  }
  return PMC_OK;
}

ResQueue res_queue(pmc_ctx *c) {
  ResQueue r; r.q = c->qres.q; r.za = c->d_resza.p; r.px = c->d_resp.p; r.py = c->d_resp.p + c->qcap; r.pz = c->d_resp.p + 2ull * c->qcap;
  return r;
}

int prepare_spots(pmc_ctx *c, const pmc_spot *spots, int nspots) {
  std::vector<SpotDev> sd(nspots); std::vector<double> cdf(nspots);
  double tot = 0;
  for (int i = 0; i < nspots; ++i) { if (!(spots[i].weight >= 0)) return fail(c, PMC_E_INVALID_ARG, "negative spot weight"); tot += spots[i].weight; }
  if (!(tot > 0)) return fail(c, PMC_E_INVALID_ARG, "spot weights sum to zero");
  double acc = 0;
  for (int i = 0; i < nspots; ++i) {
    const pmc_spot &s = spots[i]; SpotDev &d = sd[i];
    double n = std::sqrt(s.dir[0] * s.dir[0] + s.dir[1] * s.dir[1] + s.dir[2] * s.dir[2]);
    if (!(n > 0)) return fail(c, PMC_E_INVALID_ARG, "zero spot direction");
    for (int k = 0; k < 3; ++k) d.ax[k] = s.dir[k] / n;
    const double a[3] = {0.0, std::fabs(d.ax[2]) >= 0.9 ? 1.0 : 0.0, std::fabs(d.ax[2]) >= 0.9 ? 0.0 : 1.0};
    double ex[3] = {a[1] * d.ax[2] - a[2] * d.ax[1], a[2] * d.ax[0] - a[0] * d.ax[2], a[0] * d.ax[1] - a[1] * d.ax[0]};
    n = std::sqrt(ex[0] * ex[0] + ex[1] * ex[1] + ex[2] * ex[2]);
    for (int k = 0; k < 3; ++k) d.ex[k] = ex[k] / n;
    d.ey[0] = d.ax[1] * d.ex[2] - d.ax[2] * d.ex[1]; d.ey[1] = d.ax[2] * d.ex[0] - d.ax[0] * d.ex[2]; d.ey[2] = d.ax[0] * d.ex[1] - d.ax[1] * d.ex[0];
    for (int k = 0; k < 3; ++k) d.pos[k] = s.pos_cm[k];
    d.e = s.e_mev; d.sigma_e = s.sigma_e_mev; d.sx = s.sigma_x_cm; d.sy = s.sigma_y_cm; d.divx = s.div_x_rad; d.divy = s.div_y_rad;
    acc += s.weight; cdf[i] = acc / tot;
  }
  cdf[nspots - 1] = 1.0;
  std::vector<uint32_t> guide(SPOT_GUIDE + 1);
  for (int j = 0, i = 0; j <= SPOT_GUIDE; ++j) {       // first spot whose cumulative weight reaches j / SPOT_GUIDE
    while (i < nspots - 1 && cdf[i] < (double)j / SPOT_GUIDE) ++i;
    guide[j] = (uint32_t)i;
  }
  CK(c->d_spots.upload(sd, c->stream)); CK(c->d_cdf.upload(cdf, c->stream)); CK(c->d_guide.upload(guide, c->stream));
  return PMC_OK;
}

// Philox4x32-10 key schedule of a seed: round r uses (seed_lo + r W0, seed_hi + r W1), the Weyl sequence of Salmon et al.
RoundKeys key_schedule(uint64_t seed) {
  RoundKeys K;
  for (int r = 0; r < 10; ++r) {
    K.k[2 * r] = (uint32_t)seed + (uint32_t)r * 0x9E3779B9u; K.k[2 * r + 1] = (uint32_t)(seed >> 32) + (uint32_t)r * 0xBB67AE85u;
  }
  return K;
}

// Always-on per-kernel-class timing: an event pair from a pool is recorded around every launch on the context's
// stream (no synchronisation); the pairs are resolved once at the end of the call, after the stream is idle.
struct Timer {
  pmc_ctx *c; size_t i; bool on;
  Timer(pmc_ctx *c_, float *a, bool on_) : c(c_), i(0), on(on_) {
    if (!on) return;
    if (c->ev_used + 2 > c->ev_pool.size()) {
      for (int k = 0; k < 64; ++k) { cudaEvent_t e = nullptr; if (cudaEventCreate(&e) != cudaSuccess) { on = false; return; } c->ev_pool.push_back(e); }
    }
    i = c->ev_used; c->ev_used += 2; c->ev_acc.push_back(a);
    cudaEventRecord(c->ev_pool[i], c->stream);
  }
  ~Timer() { if (on) cudaEventRecord(c->ev_pool[i + 1], c->stream); }
};
void resolve_timers(pmc_ctx *c) {       // stream must be idle
  for (size_t k = 0; k < c->ev_acc.size(); ++k) {
    float ms = 0;
    if (cudaEventElapsedTime(&ms, c->ev_pool[2 * k], c->ev_pool[2 * k + 1]) == cudaSuccess) *c->ev_acc[k] += ms;
  }
  c->ev_used = 0; c->ev_acc.clear();
}

// The event-based scheduler (north_star; replaces the paper's transport kernel + Thrust collect/sort, L136):
// generation loop over compacted queues until every queue is empty.  Every kernel reads the size of its input queue on
// the device, so the host does not wait between generations: it enqueues GEN_BURST generations, then reads the size of
// the next queue once (C4 and C5 need 6 generations: one wait per sub-group) and goes on only if it is not empty.
int run_generations(pmc_ctx *c, RunParams P, bool profile) {
  cudaStream_t s = c->stream;
  QueueMem *cur = &c->qa, *nxt = &c->qb;
  const int grid_t = c->n_sm * TRANSPORT_BLOCKS_PER_SM, grid_e = c->n_sm * 4;
  ResQueue rq = res_queue(c);
  uint32_t *gen_n = c->d_head.p + 4;                 // particles entering generation g (read back at the end)
  CK(cudaMemsetAsync(gen_n, 0, GEN_SLOTS * 4, s));
  int g = 0, burst = GEN_BURST;
  while (true) {
    for (int k = 0; k < burst && g < GEN_SLOTS; ++k, ++g) {
      reset_kernel<<<1, 32, 0, s>>>(c->d_head.p, nxt->q.count, c->qel.q.count, c->qne.q.count, c->qres.q.count, c->qev.q.count);
      c->timing.launches_total++;
      { Timer t(c, &c->timing.transport_ms, profile);
        const bool mol = c->T.mcs_model == 1, dbg = P.dbg_out != nullptr;
        const bool extra = !dbg && (P.let_num != nullptr || P.roi_map != nullptr || P.aggregate != 0 || P.skip_tally != 0);
#define PMC_LAUNCH_TRANSPORT(M, D, X) transport_kernel<M, D, X><<<grid_t, TRANSPORT_THREADS, c->smem_transport, s>>>(c->T, c->G, P, cur->q, gen_n + g, c->d_head.p, c->qev.q, c->d_tally.p, c->d_cnt.p)
        if (dbg) { if (mol) PMC_LAUNCH_TRANSPORT(1, true, false); else PMC_LAUNCH_TRANSPORT(0, true, false); }
        else if (mol) { if (extra) PMC_LAUNCH_TRANSPORT(1, false, true); else PMC_LAUNCH_TRANSPORT(1, false, false); }
        else { if (extra) PMC_LAUNCH_TRANSPORT(0, false, true); else PMC_LAUNCH_TRANSPORT(0, false, false); }
#undef PMC_LAUNCH_TRANSPORT
      }
      c->timing.launches_total++; c->timing.launches_transport++;
      if (P.dbg_out) { c->counters.n_generations = 1; return PMC_OK; }     // first-steps path: the primaries' generation only
      { Timer t(c, &c->timing.elastic_ms, profile);
        event_kernel<<<grid_e, 256, 0, s>>>(c->T, c->G, P, c->qev.q, c->qel.q, c->qne.q, nxt->q, c->d_cnt.p);
        elastic_kernel<<<grid_e, 256, 0, s>>>(c->T, P, c->qel.q, nxt->q, c->d_tally.p, c->d_cnt.p); }
      { Timer t(c, &c->timing.inc_ms, profile);
        inc_kernel<<<c->n_sm * c->inc_bpsm, 128, 0, s>>>(c->T, P, c->qne.q, c->d_head.p + 1, nxt->q, rq, c->d_tally.p, c->d_cnt.p); }
      { Timer t(c, &c->timing.evaporation_ms, profile);
        evap_kernel<<<c->n_sm * c->evap_bpsm, 128, 0, s>>>(c->T, P, rq, c->d_head.p + 2, nxt->q, c->d_tally.p, c->d_cnt.p); }
      c->timing.launches_total += 4;
      std::swap(cur, nxt);
    }
    CK(cudaMemcpyAsync(c->h_pinned, cur->q.count, 4, cudaMemcpyDeviceToHost, s));
    CK(cudaMemcpyAsync(c->h_pinned + 1, gen_n, GEN_SLOTS * 4, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    c->counters.n_host_waits++;
    if (c->h_pinned[0] > c->qcap) return fail(c, PMC_E_CAPACITY, "particle queue overflow (raise chunk capacity / lower chunk_histories)");
    if (c->h_pinned[0] == 0) break;
    if (g >= GEN_SLOTS) return fail(c, PMC_E_UNSUPPORTED, "more than 64 generations of secondaries");
    burst = GEN_MORE;
  }
  for (int k = 0; k < g; ++k) if (c->h_pinned[1 + k] > 0) c->counters.n_generations++;
  return PMC_OK;
}

int fetch_counters(pmc_ctx *c) {
  Counters h{};
  CK(cudaMemcpyAsync(&h, c->d_cnt.p, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  pmc_counters &o = c->counters;
  o.n_steps = h.n_steps; o.n_elastic = h.n_elastic; o.n_nonelastic = h.n_nonelastic; o.n_secondary_protons = h.n_secondary;
  o.n_missed = h.n_missed; o.n_inc_tries = h.n_inc_tries; o.n_zab_violations = h.n_zab_bad;
  o.n_inc_guard_trips = h.n_inc_guard; o.n_inc_cap_trips = h.n_inc_cap; o.inc_max_stack = h.inc_max_stack; o.inc_max_out = h.inc_max_out;
  o.e_source = h.e_source; o.e_deposit = h.e_deposit; o.e_escape = h.e_escape; o.e_neutron = h.e_neutron; o.e_gamma = h.e_gamma;
  o.e_q = h.e_q; o.e_air = h.e_air;
  if (h.overflow) { char b[96]; snprintf(b, sizeof b, "internal queue overflow (mask 0x%x)", h.overflow); return fail(c, PMC_E_CAPACITY, b); }
  return PMC_OK;
}

int air_params(pmc_ctx *c, float &rho, float &wf, float &inv_x0, float &zoa, int &table) {
  // material of HU -1000 (air between the nozzle exit and the CT volume)
  const HostMat *m = &c->mats.front();
  for (const HostMat &h : c->mats) if (-1000 >= h.b.hu_lo && -1000 < h.b.hu_hi) m = &h;
  if (-1000 >= c->mats.back().b.hu_hi) m = &c->mats.back();
  const int hh = std::min(std::max(-1000, m->b.hu_lo), m->b.hu_hi);
  const double r = m->b.rho_lo + (m->b.rho_hi - m->b.rho_lo) * (double)(hh - m->b.hu_lo) / (double)(m->b.hu_hi - m->b.hu_lo);
  rho = (float)r; wf = (float)(m->b.table_id == 0 ? r * m->b.f_m : r); inv_x0 = (float)(1.0 / m->b.x0_gcm2); zoa = (float)m->zoa; table = m->b.table_id;
  return PMC_OK;
}

int load_ct_common(pmc_ctx *c, const int16_t *hu_dev, int nx, int ny, int nz, double dx, double dy, double dz, const double *origin) {
  c->G.hu = hu_dev; c->G.nx = nx; c->G.ny = ny; c->G.nz = nz; c->G.d[0] = (float)dx; c->G.d[1] = (float)dy; c->G.d[2] = (float)dz;
  c->G.vol = (float)(dx * dy * dz);
  for (int k = 0; k < 3; ++k) { c->G.dd[k] = k == 0 ? dx : k == 1 ? dy : dz; c->G.d[k] = (float)c->G.dd[k]; }
  for (int k = 0; k < 3; ++k) c->origin[k] = origin ? origin[k] : 0.0;   // applied on the host to the spot positions
  c->have_ct = true; c->n_roi = 0; c->dij_dev = nullptr;      // a ROI belongs to the grid it was given for
  return PMC_OK;
}

}  // namespace

extern "C" {

int pmc_create_with_allocator(pmc_ctx **out, int device, void *cuda_stream, pmc_alloc_fn alloc_fn, pmc_free_fn free_fn, void *user) {
  if (!out || ((alloc_fn == nullptr) != (free_fn == nullptr))) return PMC_E_INVALID_ARG;
  *out = nullptr;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0 || device < 0 || device >= ndev) return PMC_E_CUDA;   // no CPU fallback
  if (cudaSetDevice(device) != cudaSuccess) return PMC_E_CUDA;
  std::vector<DevBufBase *> reg;
  tl_registry = &reg;
  pmc_ctx *c = new pmc_ctx();
  tl_registry = nullptr;
  c->bufs = reg;
  c->allocator.alloc = alloc_fn; c->allocator.free = free_fn; c->allocator.user = user;
  for (DevBufBase *b : c->bufs) b->A = &c->allocator;
  c->device = device; c->stream = (cudaStream_t)cuda_stream;
  float sq[NQ];                                   // square roots of the evaporation quadrature (pmc_nuclear.cuh: EVAP_SQ)
  for (int i = 0; i < NQ; ++i) sq[i] = (float)std::sqrt((double)NQ - 0.5 - i);
  if (cudaMemcpyToSymbol(EVAP_SQ, sq, sizeof(sq)) != cudaSuccess) { delete c; return PMC_E_CUDA; }
  cudaDeviceProp prop{};
  if (cudaGetDeviceProperties(&prop, device) == cudaSuccess) c->n_sm = prop.multiProcessorCount;
  *out = c;
  return PMC_OK;
}

int pmc_create(pmc_ctx **out, int device, void *cuda_stream) {
  return pmc_create_with_allocator(out, device, cuda_stream, nullptr, nullptr, nullptr);
}

void pmc_destroy(pmc_ctx *c) {
  if (!c) return;
  cudaSetDevice(c->device);
  cudaStreamSynchronize(c->stream);
  for (DevBufBase *b : c->bufs) b->release();
  if (c->h_pinned) cudaFreeHost(c->h_pinned);
  if (c->ev[0]) { cudaEventDestroy(c->ev[0]); cudaEventDestroy(c->ev[1]); }
  for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
  delete c;
}

const char *pmc_last_error(pmc_ctx *c) { return c ? c->err.c_str() : "null context"; }

int pmc_load_physics_tables(pmc_ctx *c, const pmc_tables *t) {
  if (!c || !t) return fail(c, PMC_E_INVALID_ARG, "null argument");
  if (!t->stop_mass || !t->ln_range || !t->ln_range_d2 || !t->ln_r_lo || !t->ln_r_hi || !t->ln_energy || !t->ln_energy_d2 ||
      !t->elem_z || !t->elem_a || !t->sigma_ne_mb || !t->sigma_el_mb || !t->nuclear_mass || !t->evap_k || !t->evap_c)
    return fail(c, PMC_E_INVALID_ARG, "null table pointer");
  if (t->n_e < 4 || t->n_r < 4 || t->n_sr < 1 || t->n_sr > 4 || t->n_elem < 1 || t->n_elem > PMC_MAX_ELEM || t->mass_zdim < 3 ||
      t->mass_adim < 5 || !(t->e_min > 0) || !(t->e_max > t->e_min))
    return fail(c, PMC_E_INVALID_ARG, "bad table sizes");
  cudaSetDevice(c->device);
  c->n_e = t->n_e; c->n_r = t->n_r; c->n_sr = t->n_sr; c->n_elem = t->n_elem; c->zdim = t->mass_zdim; c->adim = t->mass_adim;
  c->e_min = t->e_min; c->e_max = t->e_max;
  auto cp = [](std::vector<double> &v, const double *p, size_t n) { v.assign(p, p + n); };
  cp(c->h_lnR, t->ln_range, (size_t)c->n_sr * c->n_e); cp(c->h_lnR2, t->ln_range_d2, (size_t)c->n_sr * c->n_e);
  cp(c->h_lnrlo, t->ln_r_lo, c->n_sr); cp(c->h_lnrhi, t->ln_r_hi, c->n_sr);
  cp(c->h_lnE, t->ln_energy, (size_t)c->n_sr * c->n_r); cp(c->h_lnE2, t->ln_energy_d2, (size_t)c->n_sr * c->n_r);
  cp(c->h_sne, t->sigma_ne_mb, (size_t)c->n_elem * c->n_e); cp(c->h_sel, t->sigma_el_mb, (size_t)c->n_elem * c->n_e);
  cp(c->h_mass, t->nuclear_mass, (size_t)c->zdim * c->adim); cp(c->h_ek, t->evap_k, (size_t)6 * c->zdim); cp(c->h_ec, t->evap_c, (size_t)6 * c->zdim);
  c->ez.assign(t->elem_z, t->elem_z + c->n_elem); c->ea.assign(t->elem_a, t->elem_a + c->n_elem);
  for (int s = 0; s < c->n_sr; ++s) {
    for (int i = 1; i < c->n_e; ++i)
      if (!(c->h_lnR[(size_t)s * c->n_e + i] > c->h_lnR[(size_t)s * c->n_e + i - 1])) return fail(c, PMC_E_INVALID_ARG, "range table not monotone");
    if (!(c->h_lnrhi[s] > c->h_lnrlo[s])) return fail(c, PMC_E_INVALID_ARG, "inverse range table abscissa not increasing");
  }
  c->h_mol.clear(); c->mol_n = 0; c->mcs_model = 0;
  if (t->mol_n > 1 && t->mol_c0 && t->mol_c1 && t->mol_c2 && t->mol_dtheta > 0) {
    c->mol_n = t->mol_n; c->mol_dth = t->mol_dtheta;
    for (const double *src : {t->mol_c0, t->mol_c1, t->mol_c2}) for (int i = 0; i < t->mol_n; ++i) c->h_mol.push_back((float)src[i]);
  }
  c->e_cut = t->e_cut; c->highland = t->highland_factor; c->kappa_g = t->kappa_gauss; c->s_max = t->s_max_wet_cm; c->n_batches = t->n_batches;
  c->h_nuc.assign(c->n_elem, Nucleus{});
  for (int i = 0; i < c->n_elem; ++i) {
    if (c->ea[i] < 1 || c->ez[i] < 0 || c->ez[i] > c->ea[i]) return fail(c, PMC_E_INVALID_ARG, "bad element");
    if (h_nmass(c, c->ez[i], c->ea[i]) <= 0) return fail(c, PMC_E_INVALID_ARG, "element missing from mass table");
    if (c->ea[i] < 2) {
      // below 250 MeV only elastic NN scattering: a lone nucleon has no non-elastic channel (and no shell model)
      for (int k = 0; k < c->n_e; ++k)
        if (c->h_sne[(size_t)i * c->n_e + k] != 0.0) return fail(c, PMC_E_INVALID_ARG, "sigma_ne_mb must be zero for an element with A < 2");
    }
    if (c->ea[i] > 1) {
      if (h_nmass(c, c->ez[i] - 1, c->ea[i] - 1) <= 0 || h_nmass(c, c->ez[i], c->ea[i] - 1) <= 0)
        return fail(c, PMC_E_INVALID_ARG, "element's neighbours missing from mass table");
      c->h_nuc[i] = build_nucleus(c, c->ez[i], c->ea[i]);
    }
  }
  c->have_tables = true; c->have_mats = false; c->mats.clear(); c->tables_dirty = true;
  return sync_tables(c);
}

int pmc_set_hu_materials(pmc_ctx *c, const pmc_hu_bin *b, int n) {
  if (!c || !b || n < 1) return fail(c, PMC_E_INVALID_ARG, "null/empty materials");
  if (!c->have_tables) return fail(c, PMC_E_STATE, "load physics tables first");
  if (n > 255) return fail(c, PMC_E_UNSUPPORTED, "at most 255 HU bins");
  cudaSetDevice(c->device);
  std::vector<HostMat> mats;
  for (int i = 0; i < n; ++i) {
    if (b[i].hu_hi <= b[i].hu_lo || (i > 0 && b[i].hu_lo != b[i - 1].hu_hi)) return fail(c, PMC_E_INVALID_ARG, "bins must be sorted and contiguous");
    double sw = 0; for (int k = 0; k < PMC_MAX_ELEM; ++k) { if (b[i].w[k] < 0) return fail(c, PMC_E_INVALID_ARG, "negative mass fraction"); sw += b[i].w[k]; }
    if (std::fabs(sw - 1) > 1e-6) return fail(c, PMC_E_INVALID_ARG, "mass fractions must sum to 1");
    for (int k = c->n_elem; k < PMC_MAX_ELEM; ++k) if (b[i].w[k] != 0) return fail(c, PMC_E_INVALID_ARG, "mass fraction on an element without cross-section rows");
    if (b[i].table_id < 0 || b[i].table_id >= c->n_sr) return fail(c, PMC_E_INVALID_ARG, "bad table id");
    if (!(b[i].rho_lo > 0) || !(b[i].rho_hi > 0) || !(b[i].x0_gcm2 > 0) || (b[i].table_id == 0 && !(b[i].f_m > 0))) return fail(c, PMC_E_INVALID_ARG, "non-positive density, f_m or X0");
    HostMat m; m.b = b[i]; m.zoa = 0;
    for (int k = 0; k < c->n_elem; ++k) m.zoa += b[i].w[k] * c->ez[k] / c->ea[k];
    mats.push_back(m);
  }
  if ((long long)mats.back().b.hu_lo - mats.front().b.hu_hi > 70000) return fail(c, PMC_E_UNSUPPORTED, "HU span too large");
  c->mats = mats; c->have_mats = true; c->tables_dirty = true;
  return sync_tables(c);
}

static int check_grid(pmc_ctx *c, const void *hu, int nx, int ny, int nz, double dx, double dy, double dz) {
  if (!c || !hu) return fail(c, PMC_E_INVALID_ARG, "null argument");
  if (nx < 1 || ny < 1 || nz < 1 || !(dx > 0) || !(dy > 0) || !(dz > 0) || (double)nx * ny * nz >= 2147483648.0) return fail(c, PMC_E_INVALID_ARG, "bad grid");
  return PMC_OK;
}

int pmc_load_ct(pmc_ctx *c, const int16_t *hu_dev, int nx, int ny, int nz, double dx, double dy, double dz, const double *origin) {
  int rc = check_grid(c, hu_dev, nx, ny, nz, dx, dy, dz); if (rc) return rc;
  cudaSetDevice(c->device);
  cudaPointerAttributes attr{};
  if (cudaPointerGetAttributes(&attr, hu_dev) != cudaSuccess || (attr.type != cudaMemoryTypeDevice && attr.type != cudaMemoryTypeManaged)) {
    cudaGetLastError();
    return fail(c, PMC_E_INVALID_ARG, "pmc_load_ct needs a device pointer (use pmc_load_ct_host for host arrays)");
  }
  return load_ct_common(c, hu_dev, nx, ny, nz, dx, dy, dz, origin);
}

int pmc_load_ct_host(pmc_ctx *c, const int16_t *hu_host, int nx, int ny, int nz, double dx, double dy, double dz, const double *origin) {
  int rc = check_grid(c, hu_host, nx, ny, nz, dx, dy, dz); if (rc) return rc;
  cudaSetDevice(c->device);
  const size_t nv = (size_t)nx * ny * nz;
  CK(c->d_hu_own.alloc(nv));
  CK(cudaMemcpyAsync(c->d_hu_own.p, hu_host, nv * sizeof(int16_t), cudaMemcpyHostToDevice, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  return load_ct_common(c, c->d_hu_own.p, nx, ny, nz, dx, dy, dz, origin);
}

int pmc_set_option(pmc_ctx *c, const char *key, double v) {
  if (!c || !key) return fail(c, PMC_E_INVALID_ARG, "null argument");
  const std::string k(key);
  if (k == "straggling") c->opt_strag = v != 0; else if (k == "mcs") c->opt_mcs = v != 0;
  else if (k == "elastic") c->opt_el = v != 0; else if (k == "nonelastic") c->opt_ne = v != 0;
  else if (k == "s_max_wet_cm") c->s_max = v; else if (k == "n_batches") { if (v < 2) return fail(c, PMC_E_INVALID_ARG, "need >= 2 batches"); c->n_batches = (int)v; }
  else if (k == "chunk_histories") { if (v < 1 || v > 67108864.0) return fail(c, PMC_E_INVALID_ARG, "chunk_histories out of range"); c->chunk = (uint64_t)v; }
  else if (k == "history_offset") { if (v < 0) return fail(c, PMC_E_INVALID_ARG, "negative offset"); c->history_offset = (uint64_t)v; }
  else if (k == "dose_aggregate") c->aggregate = v != 0;
  else if (k == "dose_scoring") c->skip_tally = v == 0;
  else if (k == "profile") c->profile = v != 0;
  else if (k == "score_letd") c->score_let = v != 0;
  else if (k == "mcs_model") { if ((v != 0 && v != 1) || (v == 1 && c->mol_n < 2)) return fail(c, PMC_E_INVALID_ARG, "mcs_model: 0 or 1 (1 needs the Moliere tables)"); c->mcs_model = (int)v; }
  else return fail(c, PMC_E_INVALID_ARG, "unknown option");
  c->tables_dirty = true;
  return PMC_OK;
}

static int simulate_impl(pmc_ctx *c, const pmc_spot *spots_in, int nspots, uint64_t n, uint64_t seed, float *dose_dev, float *sigma_dev,
                         int max_steps, float *dbg_out) {
  if (!c || !spots_in || nspots < 1) return fail(c, PMC_E_INVALID_ARG, "null argument");
  if (!c->have_tables || !c->have_mats || !c->have_ct) return fail(c, PMC_E_STATE, "call order: tables, materials, ct, simulate");
  if (n >= 4294967296ull) return fail(c, PMC_E_UNSUPPORTED, "n_histories must be < 2^32 per call");
  cudaSetDevice(c->device);
  int rc = sync_tables(c); if (rc) return rc;
  const int B = dbg_out ? 1 : c->n_batches;
  if (!dbg_out && B < 2) return fail(c, PMC_E_INVALID_ARG, "need >= 2 batches");
  // PAPER.md:L134 "groups of N/10 histories": a batch without a history has no dose to average
  if (!dbg_out && n < (uint64_t)B) return fail(c, PMC_E_INVALID_ARG, "n_histories must be at least n_batches");
  // spot positions into the grid frame
  std::vector<pmc_spot> spots(spots_in, spots_in + nspots);
  for (auto &s : spots) for (int k = 0; k < 3; ++k) s.pos_cm[k] -= c->origin[k];
  rc = prepare_spots(c, spots.data(), nspots); if (rc) return rc;
  // sub-groups: equal chunks of at most chunk_histories; every chunk carries histories of all the
  // batches it spans, each batch scoring into its own tally grid (RunParams)
  const uint64_t nchunks = std::max<uint64_t>(1, (n + c->chunk - 1) / c->chunk);
  const uint64_t chunk = std::max<uint64_t>(1, (n + nchunks - 1) / nchunks);
  rc = ensure_scratch(c, chunk); if (rc) return rc;
  const size_t nvox_s = (size_t)c->G.nx * c->G.ny * c->G.nz;
  const uint32_t nvox = (uint32_t)nvox_s;
  if ((double)nvox_s * B >= 4294967296.0) return fail(c, PMC_E_UNSUPPORTED, "n_batches x voxels must be < 2^32");
  CK(c->d_tally.alloc(nvox_s * B));
  cudaStream_t s = c->stream;
  CK(cudaMemsetAsync(c->d_tally.p, 0, nvox_s * B * 4, s)); CK(cudaMemsetAsync(c->d_cnt.p, 0, sizeof(Counters), s));
  const bool roi_on = c->n_roi > 0 && !dbg_out;
  if (roi_on) {
    if (nspots >= (1 << 24)) return fail(c, PMC_E_UNSUPPORTED, "dose influence: at most 2^24 - 1 spots");
    if ((uint64_t)nspots * c->n_roi > c->dij_cap) return fail(c, PMC_E_CAPACITY, "dose influence: nspots x n_roi exceeds the capacity of dij_dev");
    CK(cudaMemsetAsync(c->dij_dev, 0, (size_t)nspots * c->n_roi * 4, s));
  }
  const bool let_on = c->score_let && !dbg_out;
  c->have_let = false;
  if (let_on) { CK(c->d_let.alloc(2 * nvox_s)); CK(cudaMemsetAsync(c->d_let.p, 0, 2 * nvox_s * 4, s)); }
  c->counters = pmc_counters{}; c->timing = pmc_timing{};
  float air_rho, air_wf, air_ix0, air_zoa; int air_tab; air_params(c, air_rho, air_wf, air_ix0, air_zoa, air_tab);
  const bool profile = c->profile;
  c->ev_used = 0; c->ev_acc.clear();
  const cudaEvent_t e0 = c->ev[0], e1 = c->ev[1];               // created once by ensure_scratch
  CK(cudaEventRecord(e0, s));
  const int grid_v = c->n_sm * 8;
  for (uint64_t cs = 0; cs < n; cs += chunk) {
    const uint32_t nc = (uint32_t)std::min<uint64_t>(chunk, n - cs);
    RunParams P{}; P.seed = seed; P.hist0 = c->history_offset + cs; P.rk = key_schedule(seed); P.n = nc; P.max_steps = max_steps; P.dbg_out = dbg_out ? dbg_out + 8ull * cs : nullptr;
    P.aggregate = c->aggregate; P.skip_tally = c->skip_tally ? 1 : 0; P.local0 = cs; P.n_total = n; P.B = (uint32_t)B; P.nvox = nvox;
    P.roi_map = roi_on ? c->d_roimap.p : nullptr; P.dij = roi_on ? c->dij_dev : nullptr; P.n_roi = roi_on ? c->n_roi : 0u;
    P.let_num = let_on ? c->d_let.p : nullptr; P.let_den = let_on ? c->d_let.p + nvox_s : nullptr;
    P.b_over_n = (float)((double)B / (double)n); P.inv_nx = 1.0f / (float)c->G.nx; P.inv_ny = 1.0f / (float)c->G.ny;
    CK(cudaMemsetAsync(c->qa.q.count, 0, 4, s));
    { Timer t(c, &c->timing.sampler_ms, profile);
      sampler_kernel<<<(int)std::min<uint32_t>((nc + 255) / 256, (uint32_t)c->n_sm * 8), 256, 0, s>>>(c->T, c->G, c->d_spots.p, c->d_cdf.p, c->d_guide.p, nspots, P, c->qa.q, c->d_cnt.p, air_rho, air_wf, air_ix0, air_zoa, air_tab); }
    c->timing.launches_total++;
    rc = run_generations(c, P, profile); if (rc) return rc;
  }
  if (!dbg_out) {                                                  // PAPER.md:L138 total and RMS dose per voxel
    { Timer t(c, &c->timing.statistics_ms, profile);
      stats_kernel<<<grid_v, 256, 0, s>>>(c->T, c->G, c->d_tally.p, dose_dev, sigma_dev, B, n, nvox); }
    c->timing.launches_total++;
  }
  if (roi_on && n > 0)
    influence_finish_kernel<<<grid_v, 256, 0, s>>>(c->T, c->G, c->d_roivox.p, c->n_roi, (uint32_t)nspots, (float)(1.0 / (double)n), c->dij_dev);
  CK(cudaEventRecord(e1, s));
  CK(cudaGetLastError());
  rc = fetch_counters(c);
  c->have_let = let_on && rc == PMC_OK;
  resolve_timers(c);
  float ms = 0; cudaEventElapsedTime(&ms, e0, e1); c->timing.total_ms = ms;
  return rc;
}

int pmc_simulate(pmc_ctx *c, const pmc_spot *spots, int nspots, uint64_t n, uint64_t seed, float *dose_dev, float *sigma_dev) {
  if (!dose_dev || !sigma_dev) return fail(c, PMC_E_INVALID_ARG, "null output");
  return simulate_impl(c, spots, nspots, n, seed, dose_dev, sigma_dev, 0, nullptr);
}

int pmc_simulate_host(pmc_ctx *c, const pmc_spot *spots, int nspots, uint64_t n, uint64_t seed, float *dose_host, float *sigma_host) {
  if (!c || !dose_host || !sigma_host) return fail(c, PMC_E_INVALID_ARG, "null output");
  if (!c->have_ct) return fail(c, PMC_E_STATE, "call order: tables, materials, ct, simulate");
  cudaSetDevice(c->device);
  const size_t nvox = (size_t)c->G.nx * c->G.ny * c->G.nz;
  CK(c->d_out.alloc(2 * nvox));
  int rc = simulate_impl(c, spots, nspots, n, seed, c->d_out.p, c->d_out.p + nvox, 0, nullptr); if (rc) return rc;
  CK(cudaMemcpyAsync(dose_host, c->d_out.p, nvox * 4, cudaMemcpyDeviceToHost, c->stream));
  CK(cudaMemcpyAsync(sigma_host, c->d_out.p + nvox, nvox * 4, cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  return PMC_OK;
}

int pmc_first_steps(pmc_ctx *c, const pmc_spot *spot, uint64_t n, uint64_t seed, int max_steps, float *out_dev) {
  if (!out_dev || max_steps < 1) return fail(c, PMC_E_INVALID_ARG, "bad argument");
  if (c) { cudaSetDevice(c->device); cudaMemsetAsync(out_dev, 0, n * 8 * sizeof(float), c->stream); }
  return simulate_impl(c, spot, 1, n, seed, nullptr, nullptr, max_steps, out_dev);
}

int pmc_nonelastic(pmc_ctx *c, int Z, int A, double e_mev, uint64_t n, uint64_t seed, pmc_secondary *out_dev, uint64_t capacity,
                   uint32_t *off_dev, uint64_t *n_out_host) {
  if (!c || !off_dev || !n_out_host || (!out_dev && capacity > 0)) return fail(c, PMC_E_INVALID_ARG, "null argument");
  if (!c->have_tables) return fail(c, PMC_E_STATE, "load physics tables first");
  if (A < 2 || h_nmass(c, Z, A) <= 0 || h_nmass(c, Z - 1, A - 1) <= 0 || h_nmass(c, Z, A - 1) <= 0) return fail(c, PMC_E_UNSUPPORTED, "unsupported target");
  if (!(e_mev > 0)) return fail(c, PMC_E_INVALID_ARG, "non-positive energy");
  cudaSetDevice(c->device);
  int rc = sync_tables(c); if (rc) return rc;
  cudaStream_t s = c->stream;
  std::vector<Nucleus> hn(1, build_nucleus(c, Z, A));
  CK(c->d_nuc1.upload(hn, s));
  const uint32_t CH = 1u << 19;
  CK(c->d_slots.alloc((size_t)CH * MAX_SEC)); CK(c->d_counts.alloc(CH)); CK(c->d_base.alloc(1)); CK(c->d_cnt.alloc(1));
  CK(c->d_res.alloc(CH)); CK(c->d_head.alloc(4));
  CK(cudaMemsetAsync(c->d_cnt.p, 0, sizeof(Counters), s)); CK(cudaMemsetAsync(c->d_base.p, 0, 8, s));
  c->counters = pmc_counters{};
  for (uint64_t ev0 = 0; ev0 < n; ev0 += CH) {
    const uint32_t nc = (uint32_t)std::min<uint64_t>(CH, n - ev0);
    CK(cudaMemsetAsync(c->d_head.p, 0, 16, s));
    const int gb = (int)std::min<uint32_t>((nc + 127) / 128, (uint32_t)c->n_sm * 6);
    nonelastic_inc_kernel<<<gb, 128, 0, s>>>(c->T, c->d_nuc1.p, (float)e_mev, key_schedule(seed), ev0, nc, c->d_head.p + 1, c->d_slots.p, c->d_counts.p, c->d_res.p, c->d_cnt.p);
    nonelastic_evap_kernel<<<gb, 128, 0, s>>>(c->T, c->d_nuc1.p, seed, ev0, nc, c->d_head.p + 2, c->d_slots.p, c->d_counts.p, c->d_res.p, c->d_cnt.p);
    scan_kernel<<<1, 1024, 0, s>>>(c->d_counts.p, nc, off_dev + ev0, c->d_base.p);
    compact_kernel<<<(nc + 255) / 256, 256, 0, s>>>(c->d_slots.p, c->d_counts.p, off_dev + ev0, nc, reinterpret_cast<SecRec *>(out_dev), capacity);
  }
  unsigned long long total = 0;
  CK(cudaMemcpyAsync(&total, c->d_base.p, 8, cudaMemcpyDeviceToHost, s));
  CK(cudaStreamSynchronize(s));
  if (total >= 4294967296ull) return fail(c, PMC_E_UNSUPPORTED, "more than 2^32 records: split the call");
  const uint32_t t32 = (uint32_t)total;
  CK(cudaMemcpyAsync(off_dev + n, &t32, 4, cudaMemcpyHostToDevice, s));
  CK(cudaStreamSynchronize(s));
  CK(cudaGetLastError());
  *n_out_host = total;
  rc = fetch_counters(c); if (rc) return rc;
  c->counters.n_nonelastic = n;
  if (total > capacity) return fail(c, PMC_E_CAPACITY, "capacity too small");
  return PMC_OK;
}

int pmc_set_dose_influence(pmc_ctx *c, const int32_t *roi_voxels_host, int n_roi, float *dij_dev, uint64_t dij_capacity) {
  if (!c || n_roi < 0) return fail(c, PMC_E_INVALID_ARG, "bad argument");
  if (n_roi == 0) { c->n_roi = 0; c->dij_dev = nullptr; c->dij_cap = 0; return PMC_OK; }
  if (!roi_voxels_host || !dij_dev || dij_capacity < (uint64_t)n_roi) return fail(c, PMC_E_INVALID_ARG, "null ROI list / output, or capacity below one row");
  if (!c->have_ct) return fail(c, PMC_E_STATE, "load the CT first");
  cudaSetDevice(c->device);
  const size_t nvox = (size_t)c->G.nx * c->G.ny * c->G.nz;
  std::vector<int32_t> map(nvox, -1), vox(roi_voxels_host, roi_voxels_host + n_roi);
  for (int j = 0; j < n_roi; ++j) {
    if (vox[j] < 0 || (size_t)vox[j] >= nvox || map[vox[j]] >= 0) return fail(c, PMC_E_INVALID_ARG, "ROI voxel out of range or repeated");
    map[vox[j]] = j;
  }
  CK(c->d_roimap.upload(map, c->stream)); CK(c->d_roivox.upload(vox, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  c->n_roi = (uint32_t)n_roi; c->dij_dev = dij_dev; c->dij_cap = dij_capacity;
  return PMC_OK;
}

int pmc_get_letd(pmc_ctx *c, float *letd_dev) {
  if (!c || !letd_dev) return fail(c, PMC_E_INVALID_ARG, "null argument");
  if (!c->have_let) return fail(c, PMC_E_STATE, "no LET_d tally: set option score_letd = 1 and call pmc_simulate");
  cudaSetDevice(c->device);
  const size_t nvox = (size_t)c->G.nx * c->G.ny * c->G.nz;
  letd_kernel<<<c->n_sm * 8, 256, 0, c->stream>>>(c->d_let.p, c->d_let.p + nvox, letd_dev, (uint32_t)nvox);
  CK(cudaStreamSynchronize(c->stream)); CK(cudaGetLastError());
  return PMC_OK;
}

int pmc_gamma_index(pmc_ctx *c, const float *ref_dev, const float *eval_dev, int nx, int ny, int nz, double dx, double dy, double dz,
                    double dd_frac, double dta_cm, double low_dose_frac, double search_cm, float *gamma_dev, double *pass_rate_host) {
  if (!c || !ref_dev || !eval_dev || !gamma_dev) return fail(c, PMC_E_INVALID_ARG, "null argument");
  if (nx < 1 || ny < 1 || nz < 1 || !(dx > 0) || !(dy > 0) || !(dz > 0) || (double)nx * ny * nz >= 2147483648.0) return fail(c, PMC_E_INVALID_ARG, "bad grid");
  if (!(dd_frac > 0) || !(dta_cm > 0) || !(low_dose_frac >= 0)) return fail(c, PMC_E_INVALID_ARG, "criteria must be positive");
  if (nz > 65535) return fail(c, PMC_E_UNSUPPORTED, "nz > 65535");
  if (!(search_cm > 0)) search_cm = 2.0 * dta_cm;
  cudaSetDevice(c->device);
  // lattice offsets inside the search sphere, nearest first (Reading R10: voxel centres, no interpolation)
  const int rx = (int)std::floor(search_cm / dx + 1e-9), ry = (int)std::floor(search_cm / dy + 1e-9), rz = (int)std::floor(search_cm / dz + 1e-9);
  if ((double)(2 * rx + 1) * (2 * ry + 1) * (2 * rz + 1) > 4.0e6) return fail(c, PMC_E_UNSUPPORTED, "search radius spans too many voxels");
  if (rx > 32767 || ry > 32767 || rz > 32767) return fail(c, PMC_E_UNSUPPORTED, "search radius of more than 32767 voxels along an axis");
  std::vector<std::pair<double, GammaOffset>> offs;
  for (int k = -rz; k <= rz; ++k) for (int j = -ry; j <= ry; ++j) for (int i = -rx; i <= rx; ++i) {
    const double d2 = (i * dx) * (i * dx) + (j * dy) * (j * dy) + (k * dz) * (k * dz);
    if (d2 > search_cm * search_cm * (1 + 1e-12)) continue;
    GammaOffset f{}; f.i = (int16_t)i; f.j = (int16_t)j; f.k = (int16_t)k; f.d2_over_dta2 = (float)(d2 / (dta_cm * dta_cm));
    offs.push_back({d2, f});
  }
  std::stable_sort(offs.begin(), offs.end(), [](const auto &a, const auto &b) { return a.first < b.first; });
  std::vector<GammaOffset> h(offs.size());
  for (size_t i = 0; i < offs.size(); ++i) h[i] = offs[i].second;
  cudaStream_t s = c->stream;
  CK(c->d_goff.upload(h, s)); CK(c->d_gscr.alloc(3));
  CK(cudaMemsetAsync(c->d_gscr.p, 0, 3 * sizeof(unsigned long long), s));
  const uint32_t nvox = (uint32_t)((size_t)nx * ny * nz);
  GammaParams G{}; G.nx = nx; G.ny = ny; G.nz = nz; G.n_off = (int)h.size(); G.inv_dd_frac = (float)(1.0 / dd_frac); G.low_dose_frac = (float)low_dose_frac;
  uint32_t *dmax_bits = reinterpret_cast<uint32_t *>(c->d_gscr.p + 2);
  gamma_max_kernel<<<c->n_sm * 8, 256, 0, s>>>(ref_dev, nvox, dmax_bits);
  const dim3 blk(32, 8, 1), grd((nx + 31) / 32, (ny + 7) / 8, nz);
  gamma_kernel<<<grd, blk, 0, s>>>(ref_dev, eval_dev, c->d_goff.p, G, dmax_bits, gamma_dev, c->d_gscr.p);
  unsigned long long cnt[2] = {0, 0};
  CK(cudaMemcpyAsync(cnt, c->d_gscr.p, sizeof(cnt), cudaMemcpyDeviceToHost, s));
  CK(cudaStreamSynchronize(s)); CK(cudaGetLastError());
  if (pass_rate_host) *pass_rate_host = cnt[0] ? (double)cnt[1] / (double)cnt[0] : 1.0;
  return PMC_OK;
}

int pmc_get_counters(pmc_ctx *c, pmc_counters *o) { if (!c || !o) return PMC_E_INVALID_ARG; *o = c->counters; return PMC_OK; }
int pmc_get_timing(pmc_ctx *c, pmc_timing *o) { if (!c || !o) return PMC_E_INVALID_ARG; *o = c->timing; return PMC_OK; }

// ---- sub-step entry points
int pmc_philox4x32_10(pmc_ctx *c, const uint32_t *in_dev, uint64_t n, uint32_t *out_dev) {
  if (!c || (n && (!in_dev || !out_dev))) return fail(c, PMC_E_INVALID_ARG, "null argument");
  cudaSetDevice(c->device);
  if (n) philox_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(in_dev, n, out_dev);
  CK(cudaStreamSynchronize(c->stream)); CK(cudaGetLastError());
  return PMC_OK;
}
static int range_impl(pmc_ctx *c, int table, const float *in, uint64_t n, float *out, int inverse) {
  if (!c || (n && (!in || !out))) return fail(c, PMC_E_INVALID_ARG, "null argument");
  if (!c->have_tables) return fail(c, PMC_E_STATE, "load physics tables first");
  if (table < 0 || table >= c->n_sr) return fail(c, PMC_E_INVALID_ARG, "bad table id");
  cudaSetDevice(c->device);
  int rc = sync_tables(c); if (rc) return rc;
  if (n) range_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(c->T, table, in, n, out, inverse);
  CK(cudaStreamSynchronize(c->stream)); CK(cudaGetLastError());
  return PMC_OK;
}
int pmc_range_of_energy(pmc_ctx *c, int table, const float *e_dev, uint64_t n, float *r_dev) { return range_impl(c, table, e_dev, n, r_dev, 0); }
int pmc_energy_of_range(pmc_ctx *c, int table, const float *r_dev, uint64_t n, float *e_dev) { return range_impl(c, table, r_dev, n, e_dev, 1); }

static int step_range_impl(pmc_ctx *c, int bin, const float *in, uint64_t n, float *out, int inverse) {
  if (!c || (n && (!in || !out))) return fail(c, PMC_E_INVALID_ARG, "null argument");
  if (!c->have_tables || !c->have_mats) return fail(c, PMC_E_STATE, "load physics tables and HU materials first");
  if (bin < 0 || bin >= (int)c->mats.size()) return fail(c, PMC_E_INVALID_ARG, "bad HU bin index");
  cudaSetDevice(c->device);
  int rc = sync_tables(c); if (rc) return rc;
  if (n) {
    CK(cudaFuncSetAttribute(step_range_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem_transport));
    const unsigned grid = (unsigned)std::min<uint64_t>((n + 255) / 256, (uint64_t)c->n_sm * 4);
    step_range_kernel<<<grid, 256, c->smem_transport, c->stream>>>(c->T, bin, in, n, out, inverse);
  }
  CK(cudaStreamSynchronize(c->stream)); CK(cudaGetLastError());
  return PMC_OK;
}
int pmc_step_range_of_energy(pmc_ctx *c, int hu_bin, const float *e_dev, uint64_t n, float *r_dev) { return step_range_impl(c, hu_bin, e_dev, n, r_dev, 0); }
int pmc_step_energy_of_range(pmc_ctx *c, int hu_bin, const float *r_dev, uint64_t n, float *e_dev) { return step_range_impl(c, hu_bin, r_dev, n, e_dev, 1); }

int pmc_straggle(pmc_ctx *c, double e, double mean, double rhoL, double zoa, uint64_t n, uint64_t seed, float *out_dev) {
  if (!c || !out_dev) return fail(c, PMC_E_INVALID_ARG, "null argument");
  if (!c->have_tables) return fail(c, PMC_E_STATE, "load physics tables first");
  cudaSetDevice(c->device);
  int rc = sync_tables(c); if (rc) return rc;
  if (n) straggle_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(c->T, (float)e, (float)mean, (float)rhoL, (float)zoa, n, seed, out_dev);
  CK(cudaStreamSynchronize(c->stream)); CK(cudaGetLastError());
  return PMC_OK;
}

}  // extern "C"

namespace pmc {
__global__ void elastic_test_kernel(int A, float M, float tk, uint64_t n, uint64_t seed, float *out) {
  const uint64_t i = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  Rng g; g.init(seed, i, 0u, 0u);
  const ElasticOut o = elastic_event(A, M, tk, g.next4());
  out[4 * i] = o.t_gev2; out[4 * i + 1] = o.T_out; out[4 * i + 2] = o.T_rec;
  out[4 * i + 3] = acosf(fminf(1.f, fmaxf(-1.f, dot(o.dir_out, o.dir_rec))));
}
}  // namespace pmc

extern "C" int pmc_elastic(pmc_ctx *c, int Z, int A, double t_mev, uint64_t n, uint64_t seed, float *out_dev) {
  if (!c || !out_dev) return fail(c, PMC_E_INVALID_ARG, "null argument");
  if (!c->have_tables) return fail(c, PMC_E_STATE, "load physics tables first");
  if (h_nmass(c, Z, A) <= 0) return fail(c, PMC_E_UNSUPPORTED, "unsupported target");
  cudaSetDevice(c->device);
  if (n) pmc::elastic_test_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(A, (float)h_nmass(c, Z, A), (float)t_mev, n, seed, out_dev);
  CK(cudaStreamSynchronize(c->stream)); CK(cudaGetLastError());
  return PMC_OK;
}

// ---- pmc_ctx_access.h: read-only facts about a context for the library's other translation units
#include "pmc_ctx_access.h"
namespace pmc {
int ctx_device(const pmc_ctx *c) { return c->device; }
cudaStream_t ctx_stream(const pmc_ctx *c) { return c->stream; }
int ctx_sm_count(const pmc_ctx *c) { return c->n_sm; }
int ctx_fail(pmc_ctx *c, int code, const char *msg) { return fail(c, code, msg); }
}  // namespace pmc
