// yee_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, obviously-correct CPU restatement of the explicit Yee FDTD leapfrog step that
// the paper's workflow rests on ("conventional FDTD", "Yee-grid [31]"),
// with the port source of Eq. 3, the port voltage / current integrals of Eq. 4
// and the DFT of those histories.  The paper prints none of
// the update equations and no PML constants; those follow the reading fixed in DESIGN.md
// ("Readings of the paper", items R1-R14 = SURVEY.md section 8(c) O1-O9/G*).
//
// Rules this file obeys:
//   * fp64 is THE oracle.  The fp32 instantiation of the same template is only the
//     "what can fp32 time stepping achieve at all" yardstick (reading R14).
//   * Triple loops over six nx*ny*nz arrays, in the order H -> E -> source -> probes -> DFT.
//     No tiling, no fusion, no reordering.  OpenMP only on the outermost k loop.
//   * It shares no code, header, table or constant generator with the CUDA path under
//     paper_2208_04371_b200/csrc/.  Only tests/, __graft_entry__.smoke() and bench.py's
//     cpu_baseline / --impl reference legs may load it.
//
// Pins (tests/test_oracle_*.py, all "-m 'not gpu'"): CFL values the paper prints, exact discrete
// cavity eigenmode, leapfrog energy invariant, lossy-cavity recurrence, parallel-plate impedance
// eta0*d/w, Yee numerical dispersion through the V/I/DFT/S* chain, brute-force DFT, CPML
// reflection level, an independent whole-array numpy formulation on tiny grids.
// Unpinned choices (CPML grading constants, generator geometry) are listed in DESIGN.md.

#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <string>
#include <vector>

namespace {

// R2: constants chosen so that c is exact.
constexpr double kC0 = 299792458.0;
constexpr double kPi = 3.14159265358979323846264338327950288;
constexpr double kMu0 = 4.0e-7 * kPi;
constexpr double kEps0 = 1.0 / (kMu0 * kC0 * kC0);
constexpr double kEta0 = kMu0 * kC0;

enum { W_DGAUSS = 0, W_GAUSS = 1, W_GSINE = 2 };

// R6.  u = (t - t0)/sigma.
//   DGAUSS: Eq. 3, PAPER.md:50   g = -2 u exp(-u^2)
//   GAUSS :                      g = exp(-u^2)          (note exp(-u^2), not exp(-u^2/2): PAPER.md:53 f_p)
//   GSINE :                      g = sin(2 pi f0 (t - t0)) exp(-u^2)
double waveform(int kind, double t, double t0, double sigma, double f0) {
  const double u = (t - t0) / sigma;
  switch (kind) {
    case W_DGAUSS: return -2.0 * u * std::exp(-u * u);
    case W_GAUSS: return std::exp(-u * u);
    case W_GSINE: return std::sin(2.0 * kPi * f0 * (t - t0)) * std::exp(-u * u);
  }
  return 0.0;
}

struct Port {
  int has_source;
  int is, sj0, sj1, sk0, sk1;  // source box on plane i = is: columns sj0..sj1 incl., k in [sk0, sk1)
  int waveform;
  double amp, t0, sigma, f0;
  int ip;                      // probe plane
  int vj0, vj1, vk0, vk1;      // V box: columns vj0..vj1 incl., k in [vk0, vk1)
  int lj0, lj1, lk0, lk1;      // I loop encloses node columns lj0..lj1, planes lk0..lk1
};

struct Base {
  virtual ~Base() {}
  virtual void commit() = 0;
  virtual void step(long n) = 0;
  virtual void read_field(int comp, double* dst) const = 0;
  virtual void write_field(int comp, const double* src) = 0;
  virtual void read_psi_norms(double* out12) const = 0;
  virtual void read_cpml_profile(int axis, int which, double* out_n) const = 0;

  int nx = 0, ny = 0, nz = 0;
  double dx = 0, dy = 0, dz = 0, dt = 0;
  int periodic_y = 0;  // oracle-only option used by the parallel-plate pins
  int track_max = 0;
  int npml[6] = {0, 0, 0, 0, 0, 0};
  // R4 defaults: m, m_a, kappa_max, alpha_max, sigma_factor, eps_r_pml
  double cpml[6] = {3.0, 1.0, 1.0, 0.0, 0.8, 1.0};
  std::vector<double> eps[3], sig[3], mu[3];  // per component, per cell (component-sampled)
  std::vector<Port> ports;
  std::vector<double> freqs;
  std::vector<double> dftV, dftI;  // [port][freq][re,im]
  std::vector<double> lastV, lastI;
  long nstep = 0;
  double emax = 0, hmax = 0;
  bool committed = false;
  std::string err;
};

template <typename T>
struct Oracle : Base {
  std::vector<T> F[6];              // Ex Ey Ez Hx Hy Hz, index i + nx*(j + ny*k)   (R1 / SURVEY O1)
  std::vector<T> Ca[3], Cb[3], Db[3];
  // CPML per-axis profile vectors, E-profile at integer positions, H-profile at half-integer.
  std::vector<T> bE[3], cE[3], ikE[3], bH[3], cH[3], ikH[3];
  // psi arrays on slabs only.  psiH[axis][which]: the two H components transverse to axis.
  // naming: psiHxy = psi for Hx driven by d/dy, etc.
  std::vector<T> psiHxy, psiHxz, psiHyz, psiHyx, psiHzx, psiHzy;
  std::vector<T> psiExy, psiExz, psiEyz, psiEyx, psiEzx, psiEzy;
  int S[3] = {0, 0, 0};  // slab thickness lo+hi per axis

  size_t N() const { return (size_t)nx * ny * nz; }
  inline size_t id(int i, int j, int k) const { return (size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * k); }
  int n_of(int a) const { return a == 0 ? nx : (a == 1 ? ny : nz); }
  double d_of(int a) const { return a == 0 ? dx : (a == 1 ? dy : dz); }

  // slab coordinate of index u along axis a, or -1 when u is in the interior.
  inline int slab(int a, int u) const {
    const int n = n_of(a), lo = npml[2 * a], hi = npml[2 * a + 1];
    if (u < lo) return u;
    if (u >= n - hi) return lo + (u - (n - hi));
    return -1;
  }
  inline size_t px(int s, int j, int k) const { return (size_t)s + (size_t)S[0] * ((size_t)j + (size_t)ny * k); }
  inline size_t py(int i, int s, int k) const { return (size_t)i + (size_t)nx * ((size_t)s + (size_t)S[1] * k); }
  inline size_t pz(int i, int j, int s) const { return (size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * s); }

  // out-of-range operands are 0 (PEC wall behind everything); optional wrap in y.
  inline T at(int c, int i, int j, int k) const {
    if (periodic_y) { if (j < 0) j += ny; else if (j >= ny) j -= ny; }
    if (i < 0 || i >= nx || j < 0 || j >= ny || k < 0 || k >= nz) return T(0);
    return F[c][id(i, j, k)];
  }

  void commit() override {
    const size_t n = N();
    for (int c = 0; c < 6; ++c) F[c].assign(n, T(0));
    // R3: semi-implicit conductivity.  a = sigma dt / (2 eps0 eps_r)
    //   Ca = (1-a)/(1+a), Cb = (dt/(eps0 eps_r))/(1+a); sigma = +inf => Ca = Cb = 0 (PEC)
    //   Db = dt/(mu0 mu_r)
    for (int c = 0; c < 3; ++c) {
      Ca[c].resize(n); Cb[c].resize(n); Db[c].resize(n);
      for (size_t q = 0; q < n; ++q) {
        const double er = eps[c][q], sg = sig[c][q], mr = mu[c].empty() ? 1.0 : mu[c][q];
        if (std::isinf(sg)) { Ca[c][q] = T(0); Cb[c][q] = T(0); }
        else {
          const double a = sg * dt / (2.0 * kEps0 * er);
          Ca[c][q] = T((1.0 - a) / (1.0 + a));
          Cb[c][q] = T((dt / (kEps0 * er)) / (1.0 + a));
        }
        Db[c][q] = T(dt / (kMu0 * mr));
      }
    }
    // R4: CPML grading.
    const double m = cpml[0], ma = cpml[1], kmax = cpml[2], amax = cpml[3], sfac = cpml[4], erp = cpml[5];
    for (int a = 0; a < 3; ++a) {
      const int nn = n_of(a), lo = npml[2 * a], hi = npml[2 * a + 1];
      S[a] = lo + hi;
      const double smax = sfac * (m + 1.0) / (kEta0 * d_of(a) * std::sqrt(erp));
      bE[a].assign(nn, T(1)); cE[a].assign(nn, T(0)); ikE[a].assign(nn, T(1));
      bH[a].assign(nn, T(1)); cH[a].assign(nn, T(0)); ikH[a].assign(nn, T(1));
      for (int u = 0; u < nn; ++u) {
        for (int half = 0; half < 2; ++half) {
          const double pos = u + 0.5 * half;
          double rho = 0.0;
          if (lo > 0 && pos < lo) rho = (lo - pos) / lo;
          else if (hi > 0 && pos > nn - hi) rho = (pos - (nn - hi)) / hi;
          const bool in_slab = (slab(a, u) >= 0);
          if (!in_slab) continue;
          const double sg = smax * std::pow(rho, m);
          const double kp = 1.0 + (kmax - 1.0) * std::pow(rho, m);
          const double al = amax * std::pow(1.0 - rho, ma);
          const double b = std::exp(-(sg / kp + al) * dt / kEps0);
          const double den = kp * (sg + kp * al);
          const double c = (sg == 0.0) ? 0.0 : sg * (b - 1.0) / den;
          if (half == 0) { bE[a][u] = T(b); cE[a][u] = T(c); ikE[a][u] = T(1.0 / kp); }
          else           { bH[a][u] = T(b); cH[a][u] = T(c); ikH[a][u] = T(1.0 / kp); }
        }
      }
    }
    const size_t sx = (size_t)S[0] * ny * nz, sy = (size_t)nx * S[1] * nz, sz = (size_t)nx * ny * S[2];
    psiHyx.assign(sx, T(0)); psiHzx.assign(sx, T(0)); psiEyx.assign(sx, T(0)); psiEzx.assign(sx, T(0));
    psiHxy.assign(sy, T(0)); psiHzy.assign(sy, T(0)); psiExy.assign(sy, T(0)); psiEzy.assign(sy, T(0));
    psiHxz.assign(sz, T(0)); psiHyz.assign(sz, T(0)); psiExz.assign(sz, T(0)); psiEyz.assign(sz, T(0));
    dftV.assign(ports.size() * freqs.size() * 2, 0.0);
    dftI.assign(ports.size() * freqs.size() * 2, 0.0);
    lastV.assign(ports.size(), 0.0);
    lastI.assign(ports.size(), 0.0);
    nstep = 0; emax = 0; hmax = 0;
    committed = true;
  }

  // ---- R5 step 1: psi_H then H, time n+1/2 -------------------------------------
  void update_H() {
    const T idx = T(1.0 / dx), idy = T(1.0 / dy), idz = T(1.0 / dz);
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k) {
      const int sk = slab(2, k);
      for (int j = 0; j < ny; ++j) {
        const int sj = slab(1, j);
        for (int i = 0; i < nx; ++i) {
          const int si = slab(0, i);
          const size_t q = id(i, j, k);
          const T ex = F[0][q], ey = F[1][q], ez = F[2][q];
          // forward differences D+
          const T dyEz = (at(2, i, j + 1, k) - ez) * idy;
          const T dzEy = (at(1, i, j, k + 1) - ey) * idz;
          const T dzEx = (at(0, i, j, k + 1) - ex) * idz;
          const T dxEz = (at(2, i + 1, j, k) - ez) * idx;
          const T dxEy = (at(1, i + 1, j, k) - ey) * idx;
          const T dyEx = (at(0, i, j + 1, k) - ex) * idy;
          T pHxy = 0, pHxz = 0, pHyz = 0, pHyx = 0, pHzx = 0, pHzy = 0;
          if (sj >= 0) {
            const size_t p = py(i, sj, k);
            pHxy = psiHxy[p] = bH[1][j] * psiHxy[p] + cH[1][j] * dyEz;
            pHzy = psiHzy[p] = bH[1][j] * psiHzy[p] + cH[1][j] * dyEx;
          }
          if (sk >= 0) {
            const size_t p = pz(i, j, sk);
            pHxz = psiHxz[p] = bH[2][k] * psiHxz[p] + cH[2][k] * dzEy;
            pHyz = psiHyz[p] = bH[2][k] * psiHyz[p] + cH[2][k] * dzEx;
          }
          if (si >= 0) {
            const size_t p = px(si, j, k);
            pHyx = psiHyx[p] = bH[0][i] * psiHyx[p] + cH[0][i] * dxEz;
            pHzx = psiHzx[p] = bH[0][i] * psiHzx[p] + cH[0][i] * dxEy;
          }
          F[3][q] -= Db[0][q] * (dyEz * ikH[1][j] + pHxy - dzEy * ikH[2][k] - pHxz);
          F[4][q] -= Db[1][q] * (dzEx * ikH[2][k] + pHyz - dxEz * ikH[0][i] - pHyx);
          F[5][q] -= Db[2][q] * (dxEy * ikH[0][i] + pHzx - dyEx * ikH[1][j] - pHzy);
        }
      }
    }
  }

  // ---- R5 step 2: psi_E then E, time n+1; then wall rows forced to 0 ------------
  void update_E() {
    const T idx = T(1.0 / dx), idy = T(1.0 / dy), idz = T(1.0 / dz);
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k) {
      const int sk = slab(2, k);
      for (int j = 0; j < ny; ++j) {
        const int sj = slab(1, j);
        for (int i = 0; i < nx; ++i) {
          const int si = slab(0, i);
          const size_t q = id(i, j, k);
          const T hx = F[3][q], hy = F[4][q], hz = F[5][q];
          // backward differences D-
          const T dyHz = (hz - at(5, i, j - 1, k)) * idy;
          const T dzHy = (hy - at(4, i, j, k - 1)) * idz;
          const T dzHx = (hx - at(3, i, j, k - 1)) * idz;
          const T dxHz = (hz - at(5, i - 1, j, k)) * idx;
          const T dxHy = (hy - at(4, i - 1, j, k)) * idx;
          const T dyHx = (hx - at(3, i, j - 1, k)) * idy;
          T pExy = 0, pExz = 0, pEyz = 0, pEyx = 0, pEzx = 0, pEzy = 0;
          if (sj >= 0) {
            const size_t p = py(i, sj, k);
            pExy = psiExy[p] = bE[1][j] * psiExy[p] + cE[1][j] * dyHz;
            pEzy = psiEzy[p] = bE[1][j] * psiEzy[p] + cE[1][j] * dyHx;
          }
          if (sk >= 0) {
            const size_t p = pz(i, j, sk);
            pExz = psiExz[p] = bE[2][k] * psiExz[p] + cE[2][k] * dzHy;
            pEyz = psiEyz[p] = bE[2][k] * psiEyz[p] + cE[2][k] * dzHx;
          }
          if (si >= 0) {
            const size_t p = px(si, j, k);
            pEyx = psiEyx[p] = bE[0][i] * psiEyx[p] + cE[0][i] * dxHz;
            pEzx = psiEzx[p] = bE[0][i] * psiEzx[p] + cE[0][i] * dxHy;
          }
          T ex = Ca[0][q] * F[0][q] + Cb[0][q] * (dyHz * ikE[1][j] + pExy - dzHy * ikE[2][k] - pExz);
          T ey = Ca[1][q] * F[1][q] + Cb[1][q] * (dzHx * ikE[2][k] + pEyz - dxHz * ikE[0][i] - pEyx);
          T ez = Ca[2][q] * F[2][q] + Cb[2][q] * (dxHy * ikE[0][i] + pEzx - dyHx * ikE[1][j] - pEzy);
          // low-face tangential E is stored and forced to zero (PEC walls; PAPER.md:46 for the ground)
          const bool wj = (j == 0) && !periodic_y;
          if (wj || k == 0) ex = T(0);
          if (i == 0 || k == 0) ey = T(0);
          if (i == 0 || wj) ez = T(0);
          F[0][q] = ex; F[1][q] = ey; F[2][q] = ez;
        }
      }
    }
  }

  // ---- R5 step 3 (PAPER.md:53 soft source) ---------------------------------------
  void add_sources() {
    const double t = (double)(nstep + 1) * dt;
    for (const Port& p : ports) {
      if (!p.has_source) continue;
      const double g = p.amp * waveform(p.waveform, t, p.t0, p.sigma, p.f0);
      for (int k = p.sk0; k < p.sk1; ++k)
        for (int j = p.sj0; j <= p.sj1; ++j) F[2][id(p.is, j, k)] += T(g);
    }
  }

  // ---- R5 step 4, R7, R8 (Eq. 4; DFT PAPER.md:31,41) ------------
  void probes_and_dft() {
    const double tE = (double)(nstep + 1) * dt, tH = ((double)nstep + 0.5) * dt;
    for (size_t ip = 0; ip < ports.size(); ++ip) {
      const Port& p = ports[ip];
      double sv = 0.0;
      for (int j = p.vj0; j <= p.vj1; ++j)
        for (int k = p.vk0; k < p.vk1; ++k) sv += (double)F[2][id(p.ip, j, k)];
      const double V = dz / (double)(p.vj1 - p.vj0 + 1) * sv;
      double sz = 0.0, sy = 0.0;
      for (int k = p.lk0; k <= p.lk1; ++k)
        sz += (double)F[5][id(p.ip, p.lj1, k)] - (double)F[5][id(p.ip, p.lj0 - 1, k)];
      for (int j = p.lj0; j <= p.lj1; ++j)
        sy += (double)F[4][id(p.ip, j, p.lk1)] - (double)F[4][id(p.ip, j, p.lk0 - 1)];
      const double I = dz * sz - dy * sy;
      lastV[ip] = V; lastI[ip] = I;
      for (size_t m = 0; m < freqs.size(); ++m) {
        const double aE = 2.0 * kPi * freqs[m] * tE, aH = 2.0 * kPi * freqs[m] * tH;
        double* v = &dftV[(ip * freqs.size() + m) * 2];
        double* c = &dftI[(ip * freqs.size() + m) * 2];
        v[0] += V * std::cos(aE) * dt; v[1] -= V * std::sin(aE) * dt;
        c[0] += I * std::cos(aH) * dt; c[1] -= I * std::sin(aH) * dt;
      }
    }
  }

  void update_max() {
    double e = 0, h = 0;
    const size_t n = N();
    for (int c = 0; c < 3; ++c) {
      const T* a = F[c].data(); const T* b = F[c + 3].data();
#pragma omp parallel for reduction(max : e, h) schedule(static)
      for (long q = 0; q < (long)n; ++q) {
        const double x = std::fabs((double)a[q]), y = std::fabs((double)b[q]);
        if (x > e) e = x;
        if (y > h) h = y;
      }
    }
    if (e > emax) emax = e;
    if (h > hmax) hmax = h;
  }

  void step(long n) override {
    for (long s = 0; s < n; ++s) {
      update_H();
      update_E();
      add_sources();
      probes_and_dft();
      if (track_max) update_max();
      ++nstep;
    }
  }

  void read_field(int comp, double* dst) const override {
    const size_t n = N();
    for (size_t q = 0; q < n; ++q) dst[q] = (double)F[comp][q];
  }
  void write_field(int comp, const double* src) override {
    const size_t n = N();
    for (size_t q = 0; q < n; ++q) F[comp][q] = (T)src[q];
  }
  // which: 0 bE, 1 cE, 2 1/kappaE (integer positions), 3 bH, 4 cH, 5 1/kappaH (half-integer positions); n_of(axis) values
  void read_cpml_profile(int a, int which, double* out) const override {
    const std::vector<T>* v[6] = {&bE[a], &cE[a], &ikE[a], &bH[a], &cH[a], &ikH[a]};
    for (int u = 0; u < n_of(a); ++u) out[u] = (double)(*v[which])[u];
  }
  void read_psi_norms(double* out) const override {
    const std::vector<T>* v[12] = {&psiHxy, &psiHxz, &psiHyz, &psiHyx, &psiHzx, &psiHzy,
                                   &psiExy, &psiExz, &psiEyz, &psiEyx, &psiEzx, &psiEzy};
    for (int a = 0; a < 12; ++a) {
      double s = 0;
      for (T x : *v[a]) s += (double)x * (double)x;
      out[a] = std::sqrt(s);
    }
  }
};

}  // namespace

extern "C" {

// R2: physical constants, exposed so that tests can check them against CODATA-exact c and mu0.
void yo_constants(double* out4) { out4[0] = kC0; out4[1] = kMu0; out4[2] = kEps0; out4[3] = kEta0; }

// A2 / P1: the CFL limit dt_max = 1/(c sqrt(1/dx^2 + 1/dy^2 + 1/dz^2)).
double yo_cfl_dt(double dx, double dy, double dz) {
  return 1.0 / (kC0 * std::sqrt(1.0 / (dx * dx) + 1.0 / (dy * dy) + 1.0 / (dz * dz)));
}

double yo_waveform(int kind, double t, double t0, double sigma, double f0) {
  return waveform(kind, t, t0, sigma, f0);
}

void* yo_create(int nx, int ny, int nz, double dx, double dy, double dz, double dt, int use_f32,
                int periodic_y) {
  if (nx < 2 || ny < 2 || nz < 2 || !(dx > 0) || !(dy > 0) || !(dz > 0) || !(dt > 0)) return nullptr;
  if (dt > yo_cfl_dt(dx, dy, dz)) return nullptr;
  Base* b = use_f32 ? static_cast<Base*>(new Oracle<float>()) : static_cast<Base*>(new Oracle<double>());
  b->nx = nx; b->ny = ny; b->nz = nz; b->dx = dx; b->dy = dy; b->dz = dz; b->dt = dt;
  b->periodic_y = periodic_y;
  return b;
}

void yo_destroy(void* h) { delete static_cast<Base*>(h); }

int yo_set_boundary(void* h, const int* pml6, const double* cpml6) {
  Base* b = static_cast<Base*>(h);
  for (int a = 0; a < 3; ++a) {
    const int n = a == 0 ? b->nx : (a == 1 ? b->ny : b->nz);
    if (pml6[2 * a] < 0 || pml6[2 * a + 1] < 0 || pml6[2 * a] + pml6[2 * a + 1] > n) return -1;
  }
  for (int a = 0; a < 6; ++a) b->npml[a] = pml6[a];
  if (cpml6) for (int a = 0; a < 6; ++a) b->cpml[a] = cpml6[a];
  return 0;
}

// Component-sampled material arrays (R3, R12): eps_r, sigma (and optionally mu_r) for the three
// E (resp. H) components, N doubles each.  The oracle never averages.
int yo_set_materials(void* h, const double* ex, const double* ey, const double* ez, const double* sx,
                     const double* sy, const double* sz, const double* mx, const double* my,
                     const double* mz) {
  Base* b = static_cast<Base*>(h);
  const size_t n = (size_t)b->nx * b->ny * b->nz;
  const double* e[3] = {ex, ey, ez}; const double* s[3] = {sx, sy, sz}; const double* m[3] = {mx, my, mz};
  for (int c = 0; c < 3; ++c) {
    b->eps[c].assign(e[c], e[c] + n);
    b->sig[c].assign(s[c], s[c] + n);
    if (m[c]) b->mu[c].assign(m[c], m[c] + n); else b->mu[c].clear();
  }
  return 0;
}

int yo_add_port(void* h, const int* ints18, const double* dbl4) {
  Base* b = static_cast<Base*>(h);
  Port p;
  p.has_source = ints18[0]; p.is = ints18[1]; p.sj0 = ints18[2]; p.sj1 = ints18[3]; p.sk0 = ints18[4];
  p.sk1 = ints18[5]; p.waveform = ints18[6]; p.ip = ints18[7]; p.vj0 = ints18[8]; p.vj1 = ints18[9];
  p.vk0 = ints18[10]; p.vk1 = ints18[11]; p.lj0 = ints18[12]; p.lj1 = ints18[13]; p.lk0 = ints18[14];
  p.lk1 = ints18[15];
  p.amp = dbl4[0]; p.t0 = dbl4[1]; p.sigma = dbl4[2]; p.f0 = dbl4[3];
  // range checks only: samples must exist
  auto in = [](int v, int lo, int hi) { return v >= lo && v < hi; };
  if (p.has_source && !(in(p.is, 0, b->nx) && in(p.sj0, 0, b->ny) && in(p.sj1, p.sj0, b->ny) &&
                        in(p.sk0, 0, b->nz) && p.sk1 > p.sk0 && p.sk1 <= b->nz)) return -1;
  if (!(in(p.ip, 0, b->nx) && in(p.vj0, 0, b->ny) && in(p.vj1, p.vj0, b->ny) && in(p.vk0, 0, b->nz) &&
        p.vk1 > p.vk0 && p.vk1 <= b->nz)) return -1;
  if (!(in(p.lj0, 1, b->ny) && in(p.lj1, p.lj0, b->ny) && in(p.lk0, 1, b->nz) && in(p.lk1, p.lk0, b->nz)))
    return -1;
  b->ports.push_back(p);
  return (int)b->ports.size() - 1;
}

int yo_set_dft(void* h, const double* f, int nf) {
  Base* b = static_cast<Base*>(h);
  b->freqs.assign(f, f + nf);
  return 0;
}

int yo_set_track_max(void* h, int on) { static_cast<Base*>(h)->track_max = on; return 0; }

int yo_commit(void* h) {
  Base* b = static_cast<Base*>(h);
  const size_t n = (size_t)b->nx * b->ny * b->nz;
  for (int c = 0; c < 3; ++c) {
    if (b->eps[c].empty()) { b->eps[c].assign(n, 1.0); b->sig[c].assign(n, 0.0); }
  }
  b->commit();
  return 0;
}

int yo_step(void* h, long n) {
  Base* b = static_cast<Base*>(h);
  if (!b->committed) return -3;
  b->step(n);
  return 0;
}

long yo_step_count(void* h) { return static_cast<Base*>(h)->nstep; }
int yo_read_field(void* h, int comp, double* dst) { static_cast<Base*>(h)->read_field(comp, dst); return 0; }
int yo_write_field(void* h, int comp, const double* src) { static_cast<Base*>(h)->write_field(comp, src); return 0; }

int yo_read_port_dft(void* h, int port, double* V, double* I) {
  Base* b = static_cast<Base*>(h);
  if (port < 0 || port >= (int)b->ports.size()) return -1;
  const size_t nf = b->freqs.size();
  std::memcpy(V, &b->dftV[(size_t)port * nf * 2], nf * 2 * sizeof(double));
  std::memcpy(I, &b->dftI[(size_t)port * nf * 2], nf * 2 * sizeof(double));
  return 0;
}

int yo_read_port_last(void* h, int port, double* V, double* I) {
  Base* b = static_cast<Base*>(h);
  if (port < 0 || port >= (int)b->ports.size()) return -1;
  *V = b->lastV[port]; *I = b->lastI[port];
  return 0;
}

// running maxima over space and time of |E| and |H| (reading R13 = SURVEY G20)
int yo_running_max(void* h, double* e, double* hm) {
  Base* b = static_cast<Base*>(h);
  *e = b->emax; *hm = b->hmax;
  return 0;
}

// R4: the CPML coefficient vectors of one axis as the oracle uses them (pin: tests/golden/cpml_profile_lo4_hi3.txt)
int yo_cpml_profile(void* h, int axis, int which, double* out_n) {
  Base* b = static_cast<Base*>(h);
  if (!b->committed || axis < 0 || axis > 2 || which < 0 || which > 5) return -1;
  b->read_cpml_profile(axis, which, out_n);
  return 0;
}

int yo_psi_norms(void* h, double* out12) { static_cast<Base*>(h)->read_psi_norms(out12); return 0; }

}  // extern "C"
