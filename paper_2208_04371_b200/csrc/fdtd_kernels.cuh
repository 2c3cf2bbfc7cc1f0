// fdtd_kernels.cuh -- sm_100a kernels of the two-pass Yee step (H pass, E pass) and of the port work.
//
// One leapfrog step (include/fdtd.h; R5; "conventional FDTD" on a "Yee-grid"):
//   k_update_H : psi_H on the CPML slabs, then H^{n+1/2} = H^{n-1/2} - Db * curl E^n          (all cells)
//   k_update_E : psi_E on the CPML slabs, then E^{n+1} = Ca E^n + Cb * curl H^{n+1/2}, walls   (all cells)
//   k_source   : E_z += amp * g((n+1) dt) on the source boxes (Eq. 3)
//   k_probe_dft: V, I of every port (Eq. 4) and their running DFT
// Each thread of the field kernels owns 16 bytes of consecutive x cells (float4 / double2): every aligned operand
// (own cell, y+-1 row, z+-1 plane) is one 128-bit load, the x+-1 operand is one extra scalar load that hits the same
// or the neighbouring L1 line.  The zero halo of the layout (fdtd_params.h) removes all bounds tests.
#pragma once
#include <cuda_runtime.h>
#include "fdtd_params.h"

namespace fdtd_b200 {

template <typename T> struct VecOf;
template <> struct VecOf<float>  { static constexpr int V = 4; };
template <> struct VecOf<double> { static constexpr int V = 2; };

__device__ __forceinline__ void ldv(const float* p, float (&r)[4]) {
  const float4 v = *reinterpret_cast<const float4*>(p);
  r[0] = v.x; r[1] = v.y; r[2] = v.z; r[3] = v.w;
}
__device__ __forceinline__ void ldv(const double* p, double (&r)[2]) {
  const double2 v = *reinterpret_cast<const double2*>(p);
  r[0] = v.x; r[1] = v.y;
}
__device__ __forceinline__ void stv(float* p, const float (&r)[4]) {
  *reinterpret_cast<float4*>(p) = make_float4(r[0], r[1], r[2], r[3]);
}
__device__ __forceinline__ void stv(double* p, const double (&r)[2]) {
  *reinterpret_cast<double2*>(p) = make_double2(r[0], r[1]);
}

// four consecutive table words with the widest loads the type allows (read-only path)
template <typename T> struct Vec4 { T a, b, c, d; };
__device__ __forceinline__ Vec4<float> ld4(const float* p) {
  const float4 v = __ldg(reinterpret_cast<const float4*>(p));
  return {v.x, v.y, v.z, v.w};
}
__device__ __forceinline__ Vec4<double> ld4(const double* p) {
  const double2 u = __ldg(reinterpret_cast<const double2*>(p)), w = __ldg(reinterpret_cast<const double2*>(p) + 1);
  return {u.x, u.y, w.x, w.y};
}
// the material indices of a thread's V consecutive cells in one load
template <int V> __device__ __forceinline__ void ld_index(const uint8_t* p, unsigned char (&m)[V]);
template <> __device__ __forceinline__ void ld_index<4>(const uint8_t* p, unsigned char (&m)[4]) {
  const uchar4 q = __ldg(reinterpret_cast<const uchar4*>(p));
  m[0] = q.x; m[1] = q.y; m[2] = q.z; m[3] = q.w;
}
template <> __device__ __forceinline__ void ld_index<2>(const uint8_t* p, unsigned char (&m)[2]) {
  const uchar2 q = __ldg(reinterpret_cast<const uchar2*>(p));
  m[0] = q.x; m[1] = q.y;
}

// slab coordinate of index u on an axis of n cells with lo / hi CPML cells, or -1 in the interior
__device__ __forceinline__ int slab_coord(int u, int lo, int hi, int n) {
  return u < lo ? u : (u >= n - hi ? lo + u - (n - hi) : -1);
}
// padded x-slab coordinate of cell i (fdtd_params.h: the x slabs are stored in whole vectors), or -1 outside
template <typename T>
__device__ __forceinline__ int xslab_coord(const StepParams<T>& p, int i) {
  return i < p.xlo_end ? i : (i >= p.xhi_begin ? p.xlo_end + (i - p.xhi_begin) : -1);
}

// Material modes: bit 0 = full per-cell coefficient arrays (else uint8 index + table), bit 1 = permeability given.
enum { kModeIndexed = 0, kModeFull = 1, kModeMu = 2 };

// ------------------------------------------------------------------------------------------------------------------
// H pass.  R5 step 1:  psiH = bH psiH + cH D+E ;  Hx -= Dbx (D+y Ez / kHy + psiHxy - D+z Ey / kHz - psiHxz)  etc.
// ------------------------------------------------------------------------------------------------------------------
// the H update of the V consecutive cells starting at (i0, j, k); i0 < nx, j < ny
// x slabs are stored in whole vectors (fdtd_params.h), so a thread's V cells are wholly inside or wholly outside: the x-slab
// update is 128-bit psi and coefficient accesses for any layer thickness (a cell-by-cell path cost the fused step 40 % on
// grids with 10-cell layers: profiles/r02_midsize.md).
template <typename T, int MODE>
__device__ __forceinline__ void update_H_vec(const StepParams<T>& p, int i0, int j, int k) {
  constexpr int V = VecOf<T>::V;
  const long long o = i0 + (long long)p.P * j + p.PS * k;

  T ex[V], ey[V], ez[V], exk[V], eyk[V], exj[V], ezj[V], hx[V], hy[V], hz[V];
  ldv(p.src[kEx] + o, ex); ldv(p.src[kEy] + o, ey); ldv(p.src[kEz] + o, ez);
  ldv(p.src[kEx] + o + p.PS, exk); ldv(p.src[kEy] + o + p.PS, eyk);
  ldv(p.src[kEx] + o + p.P, exj);  ldv(p.src[kEz] + o + p.P, ezj);
  const T eyi = p.src[kEy][o + V], ezi = p.src[kEz][o + V];
  ldv(p.src[kHx] + o, hx); ldv(p.src[kHy] + o, hy); ldv(p.src[kHz] + o, hz);

  const int sj = slab_coord(j, p.lo[1], p.hi[1], p.ny);
  const int sk = slab_coord(k, p.lo[2], p.hi[2], p.nz);
  const bool xs = (i0 < p.xlo_end) || (i0 >= p.xhi_begin);

  T ax[V], ay[V], az[V];          // curl accumulators
  T d0[V], d1[V], d2[V], d3[V];  // raw derivatives kept for the y / z slab psi updates
  T dxa[V], dxb[V];               // D+x Ez, D+x Ey for the vectorised x-slab update
  {
    const T iky = sj >= 0 ? p.kH[1][sj] : T(1), ikz = sk >= 0 ? p.kH[2][sk] : T(1);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const T eyp = (v + 1 < V) ? ey[v + 1] : eyi;
      const T ezp = (v + 1 < V) ? ez[v + 1] : ezi;
      const T dyEz = (ezj[v] - ez[v]) * p.idy_, dzEy = (eyk[v] - ey[v]) * p.idz_;
      const T dzEx = (exk[v] - ex[v]) * p.idz_, dxEz = (ezp - ez[v]) * p.idx_;
      const T dxEy = (eyp - ey[v]) * p.idx_,    dyEx = (exj[v] - ex[v]) * p.idy_;
      ax[v] = dyEz * iky - dzEy * ikz;
      ay[v] = dzEx * ikz;
      az[v] = -dyEx * iky;
      // x terms need the per-cell kappa: done in the x-slab branch or here with kappa = 1
      dxa[v] = dxEz; dxb[v] = dxEy;
      if (!xs) { ay[v] -= dxEz; az[v] += dxEy; }
      d0[v] = dyEz; d1[v] = dyEx; d2[v] = dzEy; d3[v] = dzEx;
    }
  }
  if (xs) {  // x slab, whole vector: psiHyx (from D+x Ez) -> Hy, psiHzx (from D+x Ey) -> Hz
    const int si0 = xslab_coord(p, i0);
    const long long q = si0 + (long long)p.Sxp * (j + (long long)p.ny * k);
    T a[V], d[V], b[V], c[V], ik[V];
    ldv(p.psi[pHyx] + q, a); ldv(p.psi[pHzx] + q, d);
    ldv(p.bH[0] + si0, b); ldv(p.cH[0] + si0, c); ldv(p.kH[0] + si0, ik);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      a[v] = b[v] * a[v] + c[v] * dxa[v]; d[v] = b[v] * d[v] + c[v] * dxb[v];
      ay[v] -= dxa[v] * ik[v] + a[v];
      az[v] += dxb[v] * ik[v] + d[v];
    }
    stv(p.psi[pHyx] + q, a); stv(p.psi[pHzx] + q, d);
  }
  if (sj >= 0) {  // y slab: psiHxy (from D+y Ez), psiHzy (from D+y Ex)
    const long long q = i0 + (long long)p.P * (sj + (long long)(p.lo[1] + p.hi[1]) * k);
    const T b = p.bH[1][sj], c = p.cH[1][sj];
    T a[V], d[V];
    ldv(p.psi[pHxy] + q, a); ldv(p.psi[pHzy] + q, d);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      a[v] = b * a[v] + c * d0[v]; d[v] = b * d[v] + c * d1[v];
      if (i0 + v >= p.nx) { a[v] = T(0); d[v] = T(0); }
      ax[v] += a[v]; az[v] -= d[v];
    }
    stv(p.psi[pHxy] + q, a); stv(p.psi[pHzy] + q, d);
  }
  if (sk >= 0) {  // z slab: psiHxz (from D+z Ey), psiHyz (from D+z Ex)
    const long long q = i0 + (long long)p.P * (j + (long long)p.ny * sk);
    const T b = p.bH[2][sk], c = p.cH[2][sk];
    T a[V], d[V];
    ldv(p.psi[pHxz] + q, a); ldv(p.psi[pHyz] + q, d);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      a[v] = b * a[v] + c * d2[v]; d[v] = b * d[v] + c * d3[v];
      if (i0 + v >= p.nx) { a[v] = T(0); d[v] = T(0); }
      ax[v] -= a[v]; ay[v] += d[v];
    }
    stv(p.psi[pHxz] + q, a); stv(p.psi[pHyz] + q, d);
  }
  // Db: uniform dt/mu0, or per entry / per cell when permeability was given
  T dbx[V], dby[V], dbz[V];
  if (MODE & kModeMu) {
    if (MODE & kModeFull) { ldv(p.Db[0] + o, dbx); ldv(p.Db[1] + o, dby); ldv(p.Db[2] + o, dbz); }
    else {
      unsigned char m[V];
      ld_index<V>(p.idx + o, m);
#pragma unroll
      for (int v = 0; v < V; ++v) {
        const Vec4<T> d = ld4(p.tab + kTabH + 4 * (int)m[v]);   // {Dbx, Dby, Dbz, -}
        dbx[v] = d.a; dby[v] = d.b; dbz[v] = d.c;
      }
    }
  } else {
#pragma unroll
    for (int v = 0; v < V; ++v) { dbx[v] = p.db0; dby[v] = p.db0; dbz[v] = p.db0; }
  }
#pragma unroll
  for (int v = 0; v < V; ++v) {
    hx[v] -= dbx[v] * ax[v]; hy[v] -= dby[v] * ay[v]; hz[v] -= dbz[v] * az[v];
    if (i0 + v >= p.nx) { hx[v] = T(0); hy[v] = T(0); hz[v] = T(0); }
  }
  stv(p.dst[kHx] + o, hx); stv(p.dst[kHy] + o, hy); stv(p.dst[kHz] + o, hz);
}

// REGION launches (fdtd_params.h): the block's region, and the first cell, row and plane of this thread in it (false = none)
template <typename T>
__device__ __forceinline__ bool region_cell(const StepParams<T>& p, int& i0, int& j, int& k) {
  int g = 0;
  for (int q = 1; q < p.nreg; ++q) g = blockIdx.x >= p.reg[q].blk0 ? q : g;
  const typename StepParams<T>::Region r = p.reg[g];
  const unsigned b = blockIdx.x - r.blk0;
  const int kk = (int)(b / (unsigned)r.bpp), v = (int)(b - (unsigned)kk * (unsigned)r.bpp) * (int)blockDim.x + (int)threadIdx.x, jr = v / r.nvx;
  i0 = r.i0 + (v - jr * r.nvx) * VecOf<T>::V; j = r.j0 + jr; k = r.k0 + kk;
  return jr < r.ny;
}

// REGION: the launch covers the boxes of cells listed in p.reg (one launch per half step of the shell)
template <typename T, int MODE, bool REGION = false>
__global__ void __launch_bounds__(128) k_update_H(const StepParams<T> p) {
  constexpr int V = VecOf<T>::V;
  if (REGION) {
    if (p.bump && blockIdx.x == 0 && threadIdx.x == 0) *p.nstep += 1;
    int i0, j, k;
    if (region_cell(p, i0, j, k)) update_H_vec<T, MODE>(p, i0, j, k);
    return;
  }
  // threads are numbered along the row vectors of a plane, rows back to back: no idle lanes when a row is not a
  // multiple of the block (the X3-shaped grid: 50 vectors per row)
  // (rows that are a whole number of blocks keep one row per blockIdx.y and skip the division)
  const int nvec = (p.nx + V - 1) / V, v = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = gridDim.y > 1 ? (int)blockIdx.y : v / nvec, i0 = (gridDim.y > 1 ? v : v - j * nvec) * V;
  const int k = blockIdx.z;
  if (blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0 && threadIdx.x == 0) *p.nstep += 1;
  if (j >= p.ny) return;
  update_H_vec<T, MODE>(p, i0, j, k);
}

// ------------------------------------------------------------------------------------------------------------------
// E pass.  R5 step 2:  psiE = bE psiE + cE D-H ;  Ex = Cax Ex + Cbx (D-y Hz / kEy + psiExy - D-z Hy / kEz - psiExz) ...
// then the low-face wall rows are forced to zero (PEC walls; PAPER.md:46 for the ground).
// ------------------------------------------------------------------------------------------------------------------
// the E update of the V consecutive cells starting at (i0, j, k); i0 < nx, j < ny
// PEER: the launch that updates E on plane 0 of a z slab also stores the new Ex, Ey into the lower neighbour's halo plane
template <typename T, int MODE, bool PEER = false>
__device__ __forceinline__ void update_E_vec(const StepParams<T>& p, int i0, int j, int k) {
  constexpr int V = VecOf<T>::V;
  const long long o = i0 + (long long)p.P * j + p.PS * k;

  T hx[V], hy[V], hz[V], hxk[V], hyk[V], hxj[V], hzj[V], ex[V], ey[V], ez[V];
  ldv(p.src[kHx] + o, hx); ldv(p.src[kHy] + o, hy); ldv(p.src[kHz] + o, hz);
  ldv(p.src[kHx] + o - p.PS, hxk); ldv(p.src[kHy] + o - p.PS, hyk);
  ldv(p.src[kHx] + o - p.P, hxj);  ldv(p.src[kHz] + o - p.P, hzj);
  const T hyi = p.src[kHy][o - 1], hzi = p.src[kHz][o - 1];
  ldv(p.src[kEx] + o, ex); ldv(p.src[kEy] + o, ey); ldv(p.src[kEz] + o, ez);
  // the material index goes out with the field loads: it heads the longest dependent chain (index -> table -> update)
  unsigned char mi[V];
  if (!(MODE & kModeFull)) ld_index<V>(p.idx + o, mi);

  const int sj = slab_coord(j, p.lo[1], p.hi[1], p.ny);
  const int sk = slab_coord(k, p.lo[2], p.hi[2], p.nz);
  const bool xs = (i0 < p.xlo_end) || (i0 >= p.xhi_begin);

  T ax[V], ay[V], az[V];
  T d0[V], d1[V], d2[V], d3[V];  // raw derivatives kept for the y / z slab psi updates
  T dxa[V], dxb[V];               // D-x Hz, D-x Hy for the vectorised x-slab update
  {
    const T iky = sj >= 0 ? p.kE[1][sj] : T(1), ikz = sk >= 0 ? p.kE[2][sk] : T(1);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const T hym = (v > 0) ? hy[v - 1] : hyi;
      const T hzm = (v > 0) ? hz[v - 1] : hzi;
      const T dyHz = (hz[v] - hzj[v]) * p.idy_, dzHy = (hy[v] - hyk[v]) * p.idz_;
      const T dzHx = (hx[v] - hxk[v]) * p.idz_, dxHz = (hz[v] - hzm) * p.idx_;
      const T dxHy = (hy[v] - hym) * p.idx_,    dyHx = (hx[v] - hxj[v]) * p.idy_;
      ax[v] = dyHz * iky - dzHy * ikz;
      ay[v] = dzHx * ikz;
      az[v] = -dyHx * iky;
      dxa[v] = dxHz; dxb[v] = dxHy;
      if (!xs) { ay[v] -= dxHz; az[v] += dxHy; }
      d0[v] = dyHz; d1[v] = dyHx; d2[v] = dzHy; d3[v] = dzHx;
    }
  }
  if (xs) {  // x slab, whole vector: psiEyx (from D-x Hz) -> Ey, psiEzx (from D-x Hy) -> Ez
    const int si0 = xslab_coord(p, i0);
    const long long q = si0 + (long long)p.Sxp * (j + (long long)p.ny * k);
    T a[V], d[V], b[V], c[V], ik[V];
    ldv(p.psi[pEyx] + q, a); ldv(p.psi[pEzx] + q, d);
    ldv(p.bE[0] + si0, b); ldv(p.cE[0] + si0, c); ldv(p.kE[0] + si0, ik);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      a[v] = b[v] * a[v] + c[v] * dxa[v]; d[v] = b[v] * d[v] + c[v] * dxb[v];
      ay[v] -= dxa[v] * ik[v] + a[v];
      az[v] += dxb[v] * ik[v] + d[v];
    }
    stv(p.psi[pEyx] + q, a); stv(p.psi[pEzx] + q, d);
  }
  if (sj >= 0) {  // y slab: psiExy (from D-y Hz), psiEzy (from D-y Hx)
    const long long q = i0 + (long long)p.P * (sj + (long long)(p.lo[1] + p.hi[1]) * k);
    const T b = p.bE[1][sj], c = p.cE[1][sj];
    T a[V], d[V];
    ldv(p.psi[pExy] + q, a); ldv(p.psi[pEzy] + q, d);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      a[v] = b * a[v] + c * d0[v]; d[v] = b * d[v] + c * d1[v];
      if (i0 + v >= p.nx) { a[v] = T(0); d[v] = T(0); }
      ax[v] += a[v]; az[v] -= d[v];
    }
    stv(p.psi[pExy] + q, a); stv(p.psi[pEzy] + q, d);
  }
  if (sk >= 0) {  // z slab: psiExz (from D-z Hy), psiEyz (from D-z Hx)
    const long long q = i0 + (long long)p.P * (j + (long long)p.ny * sk);
    const T b = p.bE[2][sk], c = p.cE[2][sk];
    T a[V], d[V];
    ldv(p.psi[pExz] + q, a); ldv(p.psi[pEyz] + q, d);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      a[v] = b * a[v] + c * d2[v]; d[v] = b * d[v] + c * d3[v];
      if (i0 + v >= p.nx) { a[v] = T(0); d[v] = T(0); }
      ax[v] -= a[v]; ay[v] += d[v];
    }
    stv(p.psi[pExz] + q, a); stv(p.psi[pEyz] + q, d);
  }
  T cax[V], cay[V], caz[V], cbx[V], cby[V], cbz[V];
  if (MODE & kModeFull) {
    ldv(p.Ca[0] + o, cax); ldv(p.Ca[1] + o, cay); ldv(p.Ca[2] + o, caz);
    ldv(p.Cb[0] + o, cbx); ldv(p.Cb[1] + o, cby); ldv(p.Cb[2] + o, cbz);
  } else {
#pragma unroll
    for (int v = 0; v < V; ++v) {   // mi: one 32-bit (16-bit) load for the thread's 4 (2) cells, issued with the field loads
      const Vec4<T> a = ld4(p.tab + 8 * (int)mi[v]);       // {Cax, Cay, Caz, Cbx}
      const Vec4<T> b = ld4(p.tab + 8 * (int)mi[v] + 4);   // {Cby, Cbz, -, -}
      cax[v] = a.a; cay[v] = a.b; caz[v] = a.c; cbx[v] = a.d; cby[v] = b.a; cbz[v] = b.b;
    }
  }
  const bool wj = (j == 0), wk = (k == 0) && !p.z_lo_open;
#pragma unroll
  for (int v = 0; v < V; ++v) {
    const bool wi = (i0 + v == 0), pad = (i0 + v >= p.nx);
    ex[v] = cax[v] * ex[v] + cbx[v] * ax[v];
    ey[v] = cay[v] * ey[v] + cby[v] * ay[v];
    ez[v] = caz[v] * ez[v] + cbz[v] * az[v];
    if (wj || wk || pad) ex[v] = T(0);
    if (wi || wk || pad) ey[v] = T(0);
    if (wi || wj || pad) ez[v] = T(0);
  }
  stv(p.dst[kEx] + o, ex); stv(p.dst[kEy] + o, ey); stv(p.dst[kEz] + o, ez);
  if (PEER && k == 0 && p.peer_E[0] != nullptr) {   // NVLink peer stores: the tangential E the slab below needs for its next H update
    const long long oq = i0 + (long long)p.P * j;
    stv(p.peer_E[0] + oq, ex); stv(p.peer_E[1] + oq, ey);
  }
}

template <typename T, int MODE, bool PEER = false, bool REGION = false>
__global__ void __launch_bounds__(128) k_update_E(const StepParams<T> p) {
  constexpr int V = VecOf<T>::V;
  if (REGION) {
    int i0, j, k;
    if (region_cell(p, i0, j, k)) update_E_vec<T, MODE, PEER>(p, i0, j, k);
    return;
  }
  const int nvec = (p.nx + V - 1) / V, v = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = gridDim.y > 1 ? (int)blockIdx.y : v / nvec, i0 = (gridDim.y > 1 ? v : v - j * nvec) * V;
  const int k = blockIdx.z;
  if (j >= p.ny) return;
  update_E_vec<T, MODE, PEER>(p, i0, j, k);
}

// ------------------------------------------------------------------------------------------------------------------
// z-slab hand-over flags (fdtd_z_link; guard cells exchanged every step).  A slab pushes its boundary
// planes into the neighbour's halo with peer stores from the kernel that computes them; what orders the neighbour's next
// kernel after those stores is a step counter in the NEIGHBOUR's memory:
//   k_z_post  (stream-ordered after the producing kernel)  fence; *peer_flag = step      release at system scope
//   k_z_wait  (stream-ordered before the consuming kernel) spin until *flag >= step      acquire at system scope
// `step` is read from the device step counter (+ add), so the same captured graph serves every replay.  The spin is
// bounded: after max_spins polls it records a time-out in *err and returns (no launch can hang the device); once *err is set
// every later wait of the slab returns at once (the run is lost anyway; the next synchronising read reports it) instead of
// spinning the full time-out again per step.
// ------------------------------------------------------------------------------------------------------------------
__global__ void k_z_post(unsigned long long* peer_flag, const long long* nstep, long long add) {
  const unsigned long long v = (unsigned long long)(*nstep + add);
  __threadfence_system();
  asm volatile("st.release.sys.global.u64 [%0], %1;" ::"l"(peer_flag), "l"(v) : "memory");
}
__global__ void k_z_wait(const unsigned long long* flag, const long long* nstep, long long add, int* err, long long max_spins) {
  const unsigned long long want = (unsigned long long)(*nstep + add);
  if (*reinterpret_cast<volatile int*>(err)) return;
  for (long long it = 0;; ++it) {
    unsigned long long v;
    asm volatile("ld.acquire.sys.global.u64 %0, [%1];" : "=l"(v) : "l"(flag) : "memory");
    if (v >= want) break;
    if (it >= max_spins) { atomicExch(err, 1); break; }
    __nanosleep(it < 64 ? 100 : 1000);
  }
}

// ------------------------------------------------------------------------------------------------------------------
// Port work.  The device step counter was already incremented by the first kernel of the step.
// ------------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ double waveform_dev(int kind, double t, double t0, double sigma, double f0) {
  const double u = (t - t0) / sigma;
  switch (kind) {
    case 0: return -2.0 * u * exp(-u * u);                                   // Eq. 3
    case 1: return exp(-u * u);
    case 2: return sin(2.0 * 3.14159265358979323846 * f0 * (t - t0)) * exp(-u * u);
  }
  return 0.0;
}

// one launch per driving port (in port order on the stream, so overlapping source boxes add up deterministically);
// one thread per source sample
template <typename T>
__global__ void __launch_bounds__(256) k_source(const PortParams<T> p, int n) {
  const PortDev q = p.ports[n];
  const int nj = q.sj1 - q.sj0 + 1, ns = nj * (q.sk1 - q.sk0);
  const int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= ns) return;
  const double t = (double)(*p.nstep) * p.dt;
  const T g = (T)(q.amp * waveform_dev(q.waveform, t, q.t0, q.sigma, q.f0));
  const int j = q.sj0 + s % nj, k = q.sk0 + s / nj;
  p.Ez[q.is + (long long)p.P * j + p.PS * k] += g;
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int s = 16; s > 0; s >>= 1) v += __shfl_xor_sync(0xffffffffu, v, s);
  return v;
}

// Port probes and running DFT.  grid (nblk, nports), 256 threads.  Block b of a port reduces its slice of the V box and of
// the I loop (warp-shuffle partial sums in fp64, a fixed sample -> thread -> block assignment) and writes one partial pair;
// the block that arrives last at the port's counter adds the partials in block order (so V, I do not depend on which block
// that is) and advances the DFT accumulators of every frequency:
//   V = (dz / n_col) * sum Ez over the V box                                             (Eq. 4 line 1, R7)
//   I = dz * sum_k (Hz[lj1,k] - Hz[lj0-1,k]) - dy * sum_j (Hy[j,lk1] - Hy[j,lk0-1])        (Eq. 4 line 2, R7)
//   V^[m] += V e^{-j 2 pi f_m n dt} dt,  I^[m] += I e^{-j 2 pi f_m (n - 1/2) dt} dt        (R8)
constexpr int kProbeThreads = 256;
constexpr int kProbeMaxBlocks = 64;
template <typename T>
__global__ void __launch_bounds__(kProbeThreads) k_probe_dft(const PortParams<T> p) {
  __shared__ double sh[2][kProbeThreads / 32];
  __shared__ double res[2];
  __shared__ int last;
  const int port = blockIdx.y, nblk = gridDim.x;
  const PortDev q = p.ports[port];
  const int nj = q.vj1 - q.vj0 + 1, nv = nj * (q.vk1 - q.vk0);
  const int gtid = blockIdx.x * kProbeThreads + threadIdx.x, gstride = nblk * kProbeThreads;
  double sv = 0.0;
  for (int s = gtid; s < nv; s += gstride) {
    const int j = q.vj0 + s % nj, k = q.vk0 + s / nj;
    sv += (double)p.Ez[q.ip + (long long)p.P * j + p.PS * k];
  }
  const int nkl = q.lk1 - q.lk0 + 1, njl = q.lj1 - q.lj0 + 1;
  double si = 0.0;
  for (int s = gtid; s < nkl + njl; s += gstride) {
    if (s < nkl) {
      const int k = q.lk0 + s;
      si += p.dz * ((double)p.Hz[q.ip + (long long)p.P * q.lj1 + p.PS * k] -
                    (double)p.Hz[q.ip + (long long)p.P * (q.lj0 - 1) + p.PS * k]);
    } else {
      const int j = q.lj0 + (s - nkl);
      si -= p.dy * ((double)p.Hy[q.ip + (long long)p.P * j + p.PS * q.lk1] -
                    (double)p.Hy[q.ip + (long long)p.P * j + p.PS * (q.lk0 - 1)]);
    }
  }
  sv = warp_sum(sv); si = warp_sum(si);
  const int w = threadIdx.x >> 5;
  if ((threadIdx.x & 31) == 0) { sh[0][w] = sv; sh[1][w] = si; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0.0, b = 0.0;
#pragma unroll
    for (int q2 = 0; q2 < kProbeThreads / 32; ++q2) { a += sh[0][q2]; b += sh[1][q2]; }
    double V = a, I = b;
    last = 1;
    if (nblk > 1) {   // small port boxes take one block per port and skip the hand-over through global memory
      double* part = p.partial + ((long long)port * kProbeMaxBlocks + blockIdx.x) * 2;
      part[0] = a; part[1] = b;
      __threadfence();
      last = (atomicAdd(p.pcount + port, 1) == nblk - 1);
      if (last) {
        __threadfence();
        V = 0.0; I = 0.0;
        const volatile double* pp = p.partial + (long long)port * kProbeMaxBlocks * 2;
        for (int b2 = 0; b2 < nblk; ++b2) { V += pp[2 * b2]; I += pp[2 * b2 + 1]; }
        p.pcount[port] = 0;   // ready for the next step (the kernel boundary orders it)
      }
    }
    if (last) {
      V *= p.dz / (double)nj;
      res[0] = V; res[1] = I;
      p.lastV[port] = V; p.lastI[port] = I;
    }
  }
  __syncthreads();
  if (!last) return;
  const double n = (double)(*p.nstep);
  for (int m2 = threadIdx.x; m2 < 2 * p.nf; m2 += kProbeThreads) {
    const bool isI = m2 >= p.nf;
    const int m = isI ? m2 - p.nf : m2;
    const double t = (isI ? n - 0.5 : n) * p.dt;
    double s, c;
    sincos(2.0 * 3.14159265358979323846 * p.freqs[m] * t, &s, &c);
    const double a = res[isI ? 1 : 0] * p.dt;
    double* acc = (isI ? p.dftI : p.dftV) + ((long long)port * p.nf + m) * 2;
    acc[0] += a * c;
    acc[1] -= a * s;
  }
}

// ------------------------------------------------------------------------------------------------------------------
// Setup kernels (not on the timed path).
// ------------------------------------------------------------------------------------------------------------------
// full mode: arrays hold eps_r (in ca) and sigma (in cb) on entry, Ca and Cb on exit (R3)
template <typename T>
__global__ void k_coef_E(T* ca, T* cb, long long n, double dt, double eps0) {
  const long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (q >= n) return;
  const double er = (double)ca[q], sg = (double)cb[q];
  if (er == 0.0) { ca[q] = T(0); cb[q] = T(0); return; }  // halo / pad cells: keep them inert
  if (isinf(sg)) { ca[q] = T(0); cb[q] = T(0); return; }
  const double a = sg * dt / (2.0 * eps0 * er);
  ca[q] = (T)((1.0 - a) / (1.0 + a));
  cb[q] = (T)((dt / (eps0 * er)) / (1.0 + a));
}
template <typename T>
__global__ void k_coef_H(T* db, long long n, double dt, double mu0) {
  const long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (q >= n) return;
  const double mr = (double)db[q];
  db[q] = mr == 0.0 ? T(0) : (T)(dt / (mu0 * mr));
}
// the device step counter, advanced on the stream where no field kernel of the step does it
__global__ void k_bump(long long* nstep, long long add) { *nstep += add; }

template <typename T>
__global__ void k_fill(T* a, long long n, T v) {
  const long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (q < n) a[q] = v;
}

}  // namespace fdtd_b200
