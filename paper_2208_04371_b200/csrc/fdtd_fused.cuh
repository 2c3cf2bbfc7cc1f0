// fdtd_fused.cuh -- the fused E+H step: one kernel advances H^{n-1/2} -> H^{n+1/2} and E^n -> E^{n+1}.
//
// Why: the two-pass step moves 73 B per cell-update (fp32, indexed materials): the H pass reads six fields and writes
// three, the E pass reads six (+1 B index) and writes three.  Both passes read the same six arrays.  Fusing them
// ("temporal blocking across the E/H half-steps", north_star item 1) reads each field once and writes each once: 49 B.
//
// How (R5 steps 1-2, same arithmetic and order as k_update_H / k_update_E):
//   * a thread block owns an (x,y) tile of TX x TY cells (TX = 32 lanes x 16 bytes) and marches along z over a chunk of
//     planes.  For plane k it needs E^n on planes k, k+1 and H^{n-1/2} on plane k, on the tile plus a one-cell halo:
//     E^{n+1}(c) needs H^{n+1/2}(c), H^{n+1/2}(c - e_a), which need E^n(c), E^n(c + e_b), E^n(c - e_a + e_b).
//   * TMA (cp.async.bulk.tensor.3d) brings, per plane, seven boxes into shared memory: Ex, Ey of plane k+1, Ez and
//     Hx, Hy, Hz of plane k (each (TX + 2 vectors) x (TY + 2 | TY + 1) with the halo, zero-filled outside the array)
//     and the uint8 index tile.  NS stages ring, one mbarrier per stage, one elected thread issues; the boxes of plane
//     k + NS are requested as soon as plane k has been read, so NS - 1 planes are in flight per SM with no register
//     cost.  This is what keeps HBM busy with one resident block per SM.
//   * H phase: warp w = 1..TY owns tile row w-1; warp 0 recomputes the halo row j = y0-1 (its Hx, Hz are the j-1
//     operands of the first owned row), warp TY+1 recomputes Hy, Hz of the halo column i = x0-1.  Plane k operands that
//     were loaded as "k+1" one iteration earlier are carried in registers, so an iteration reads only its own stage.
//     New Hx, Hz rows go to shared memory (for the row above), the halo column to a small array, Hy and the k-1 plane
//     of Hx, Hy stay in registers; the x-1 operands come from warp shuffles.
//   * one __syncthreads, then the E phase for the owned cells: coefficients from the shared-memory table (or the
//     full arrays), CPML, walls, store.
//   * results go to the OTHER field set (ping-pong): a neighbouring block may still need E^n / H^{n-1/2} of this tile
//     for its halo, so updating in place would be a race.  psi_H is double buffered for the same reason (the halo
//     recomputation reads the old value); psi_E is touched by the owner only and stays in place.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include "fdtd_kernels.cuh"
#include "fdtd_params.h"

namespace fdtd_b200 {

template <typename T>
struct FusedParams {
  CUtensorMap tm[7];     // boxes of the set being read: Ex Ey Ez Hx Hy Hz, then the uint8 material index
  StepParams<T> sp;      // src = set read, dst = set written; psi[0..5] = psi_H written, psi[6..11] = psi_E (in place)
  const T* psiH_src[6];  // psi_H read (pHxy pHzy pHxz pHyz pHyx pHzx)
  int kz;                // planes per z chunk (grid.z = ceil(nz / kz))
};

constexpr int round128(int v) { return (v + 127) / 128 * 128; }

template <typename T, int TY_, int NS_>
struct FusedCfg {
  static constexpr int V = VecOf<T>::V, TX = 32 * V, BX = TX + 2 * V, TY = TY_, NS = NS_;
  static constexpr int ROWS_E = TY + 2, ROWS_H = TY + 1;
  static constexpr int E_TX = ROWS_E * BX * (int)sizeof(T), H_TX = ROWS_H * BX * (int)sizeof(T), I_TX = TY * TX;
  static constexpr int E_B = round128(E_TX), H_B = round128(H_TX), I_B = round128(I_TX);
  static constexpr int STAGE = 3 * E_B + 3 * H_B + I_B;
  static constexpr int HN_B = 2 * 2 * ROWS_H * TX * (int)sizeof(T);   // [buffer][Hx|Hz][row][x]
  static constexpr int HC_B = round128(2 * 2 * TY * (int)sizeof(T));  // [buffer][Hy|Hz][row] at i = x0-1
  static constexpr int TAB_B = kTabWords * (int)sizeof(T);
  static constexpr int BAR_B = 128;
  static constexpr int SMEM = NS * STAGE + HN_B + HC_B + TAB_B + BAR_B;
  static constexpr int THREADS = (TY + 2) * 32;
};

// ---- mbarrier / TMA wrappers (PTX ISA: mbarrier, cp.async.bulk.tensor) ------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* b, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* b, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* b, unsigned parity) {
  unsigned ok;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n"
      : "=r"(ok) : "r"(smem_u32(b)), "r"(parity) : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, unsigned parity) {
  while (!mbar_try_wait(b, parity)) {}
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* tm, uint64_t* bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(
          smem_u32(dst)),
      "l"(reinterpret_cast<uint64_t>(tm)), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
      : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* tm) {
  asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(tm)) : "memory");
}

// shared-memory reads of a thread's V material indices and of one table record
template <int V> __device__ __forceinline__ void ld_index_smem(const unsigned char* p, unsigned char (&m)[V]);
template <> __device__ __forceinline__ void ld_index_smem<4>(const unsigned char* p, unsigned char (&m)[4]) {
  const uchar4 q = *reinterpret_cast<const uchar4*>(p);
  m[0] = q.x; m[1] = q.y; m[2] = q.z; m[3] = q.w;
}
template <> __device__ __forceinline__ void ld_index_smem<2>(const unsigned char* p, unsigned char (&m)[2]) {
  const uchar2 q = *reinterpret_cast<const uchar2*>(p);
  m[0] = q.x; m[1] = q.y;
}
__device__ __forceinline__ Vec4<float> lds4(const float* p) {
  const float4 v = *reinterpret_cast<const float4*>(p);
  return {v.x, v.y, v.z, v.w};
}
__device__ __forceinline__ Vec4<double> lds4(const double* p) {
  const double2 u = *reinterpret_cast<const double2*>(p), w = *(reinterpret_cast<const double2*>(p) + 1);
  return {u.x, u.y, w.x, w.y};
}

template <typename T> __device__ __forceinline__ void stv_stream(T* p, const T (&r)[VecOf<T>::V]);
template <> __device__ __forceinline__ void stv_stream<float>(float* p, const float (&r)[4]) {
  __stcs(reinterpret_cast<float4*>(p), make_float4(r[0], r[1], r[2], r[3]));
}
template <> __device__ __forceinline__ void stv_stream<double>(double* p, const double (&r)[2]) {
  __stcs(reinterpret_cast<double2*>(p), make_double2(r[0], r[1]));
}

// ------------------------------------------------------------------------------------------------------------------
template <typename T, int MODE, int TY, int NS>
__global__ void __launch_bounds__((TY + 2) * 32, 1) k_step_fused(const __grid_constant__ FusedParams<T> fp) {
  using C = FusedCfg<T, TY, NS>;
  constexpr int V = C::V, TX = C::TX, BX = C::BX;
  constexpr bool kFull = (MODE & kModeFull) != 0, kMu = (MODE & kModeMu) != 0;
  extern __shared__ __align__(1024) unsigned char smem[];
  T* const hn = reinterpret_cast<T*>(smem + NS * C::STAGE);
  T* const hc = reinterpret_cast<T*>(smem + NS * C::STAGE + C::HN_B);
  T* const tab = reinterpret_cast<T*>(smem + NS * C::STAGE + C::HN_B + C::HC_B);
  uint64_t* const bar = reinterpret_cast<uint64_t*>(smem + NS * C::STAGE + C::HN_B + C::HC_B + C::TAB_B);

  const StepParams<T>& p = fp.sp;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
  const int k0 = blockIdx.z * fp.kz, k1 = min(k0 + fp.kz, p.nz);
  const int nIt = k1 - k0 + 2;  // it = 0: Ex, Ey of plane k0-1 only; it = 1: H of plane k0-1; it >= 2: plane k0 + it - 2

  if (blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0 && threadIdx.x == 0) *p.nstep += 1;

  // one elected thread issues the boxes of iteration `it` into stage it % NS
  auto issue = [&](int it) {
    const int k = k0 - 2 + it, s = it % NS;
    unsigned char* st = smem + s * C::STAGE;
    const bool want_idx = !kFull && it >= 2;
    const unsigned bytes = it == 0 ? 2u * C::E_TX : 3u * C::E_TX + 3u * C::H_TX + (want_idx ? (unsigned)C::I_TX : 0u);
    mbar_expect_tx(&bar[s], bytes);
    tma_load_3d(st, &fp.tm[kEx], &bar[s], x0 - V, y0 - 1, k + 2);               // plane k+1 (array plane index + 1)
    tma_load_3d(st + C::E_B, &fp.tm[kEy], &bar[s], x0 - V, y0 - 1, k + 2);
    if (it >= 1) {
      tma_load_3d(st + 2 * C::E_B, &fp.tm[kEz], &bar[s], x0 - V, y0 - 1, k + 1);  // plane k
      tma_load_3d(st + 3 * C::E_B, &fp.tm[kHx], &bar[s], x0 - V, y0 - 1, k + 1);
      tma_load_3d(st + 3 * C::E_B + C::H_B, &fp.tm[kHy], &bar[s], x0 - V, y0 - 1, k + 1);
      tma_load_3d(st + 3 * C::E_B + 2 * C::H_B, &fp.tm[kHz], &bar[s], x0 - V, y0 - 1, k + 1);
      if (want_idx) tma_load_3d(st + 3 * C::E_B + 3 * C::H_B, &fp.tm[6], &bar[s], x0, y0, k + 1);
    }
  };

  if (threadIdx.x == 0) {
    for (int s = 0; s < NS; ++s) mbar_init(&bar[s], 1);
    mbar_fence_init();
#pragma unroll
    for (int q = 0; q < 7; ++q) tma_prefetch_desc(&fp.tm[q]);
  }
  if (!kFull) {
    for (int q = threadIdx.x; q < (kMu ? kTabWords : kTabH); q += C::THREADS) tab[q] = p.tab[q];
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int it = 0; it < NS && it < nIt; ++it) issue(it);
  }

  const bool rowwarp = w <= TY;
  // row warps: j = y0-1+w (w = 0 is the halo row); column warp: lane l <-> row y0+l at i = x0-1
  const int j = rowwarp ? y0 - 1 + w : y0 + lane;
  const int i0 = rowwarp ? x0 + lane * V : x0 - 1;
  const bool jin = j >= 0 && j < p.ny;
  const bool cin = rowwarp ? (jin && i0 < p.nx) : (jin && i0 >= 0 && lane < TY);  // thread's cell(s) exist
  const bool owned = rowwarp && w >= 1 && cin;
  const int sj = jin ? slab_coord(j, p.lo[1], p.hi[1], p.ny) : -1;
  const int Sx = p.lo[0] + p.hi[0], Sy = p.lo[1] + p.hi[1];
  const T iky_H = sj >= 0 ? p.kH[1][sj] : T(1), iky_E = sj >= 0 ? p.kE[1][sj] : T(1);
  const T bHy = sj >= 0 ? p.bH[1][sj] : T(0), cHy = sj >= 0 ? p.cH[1][sj] : T(0);
  const T bEy = sj >= 0 ? p.bE[1][sj] : T(0), cEy = sj >= 0 ? p.cE[1][sj] : T(0);
  const bool xs = rowwarp && ((i0 < p.lo[0]) || (i0 + V > p.nx - p.hi[0]));  // some cell of the vector is in an x slab

  // registers carried from one plane to the next
  T ex0[V], ey0[V], exj0[V], hxm[V], hym[V];
  T eyi0 = T(0);
#pragma unroll
  for (int v = 0; v < V; ++v) { ex0[v] = ey0[v] = exj0[v] = hxm[v] = hym[v] = T(0); }
  T c_ex0 = T(0), c_exj0 = T(0), c_ey0 = T(0), c_eyp0 = T(0);  // column warp: Ex(x0-1,j), Ex(x0-1,j+1), Ey(x0-1,j), Ey(x0,j)

  for (int it = 0; it < nIt; ++it) {
    const int k = k0 - 2 + it, s = it % NS;
    const unsigned char* st = smem + s * C::STAGE;
    const T* sEx = reinterpret_cast<const T*>(st);
    const T* sEy = reinterpret_cast<const T*>(st + C::E_B);
    const T* sEz = reinterpret_cast<const T*>(st + 2 * C::E_B);
    const T* sHx = reinterpret_cast<const T*>(st + 3 * C::E_B);
    const T* sHy = reinterpret_cast<const T*>(st + 3 * C::E_B + C::H_B);
    const T* sHz = reinterpret_cast<const T*>(st + 3 * C::E_B + 2 * C::H_B);
    const unsigned char* sIdx = st + 3 * C::E_B + 3 * C::H_B;
    const bool kin = k >= 0;  // k < nz always
    const int sk = kin ? slab_coord(k, p.lo[2], p.hi[2], p.nz) : -1;
    const long long o = (long long)i0 + (long long)p.P * j + p.PS * k;
    T* const hnb = hn + (it & 1) * (2 * C::ROWS_H * TX);
    T* const hcb = hc + (it & 1) * (2 * TY);

    mbar_wait(&bar[s], (unsigned)(it / NS) & 1u);

    T hx[V], hy[V], hz[V], ez[V];
    unsigned char mi[V];
    if (rowwarp) {
      // ---------------- H phase, row warps -------------------------------------------------------------------------
      const int off = w * BX + V + lane * V;
      T ex1[V], ey1[V], exj1[V];
      ldv(sEx + off, ex1); ldv(sEy + off, ey1); ldv(sEx + off + BX, exj1);
      T eyi1 = __shfl_down_sync(0xffffffffu, ey1[0], 1);
      if (lane == 31) eyi1 = sEy[off + V];
      if (it >= 1) {
        T ezj[V];
        ldv(sEz + off, ez); ldv(sEz + off + BX, ezj);
        T ezi = __shfl_down_sync(0xffffffffu, ez[0], 1);
        if (lane == 31) ezi = sEz[off + V];
        ldv(sHx + off, hx); ldv(sHy + off, hy); ldv(sHz + off, hz);
        if (!kFull && it >= 2 && w >= 1) ld_index_smem<V>(sIdx + (w - 1) * TX + lane * V, mi);

        const bool live = cin && kin;
        const T ikz = sk >= 0 ? p.kH[2][sk] : T(1);
        T ax[V], ay[V], az[V], d0[V], d1[V], d2[V], d3[V];
#pragma unroll
        for (int v = 0; v < V; ++v) {
          const T eyp = (v + 1 < V) ? ey0[v + 1] : eyi0;
          const T ezp = (v + 1 < V) ? ez[v + 1] : ezi;
          const T dyEz = (ezj[v] - ez[v]) * p.idy_, dzEy = (ey1[v] - ey0[v]) * p.idz_;
          const T dzEx = (ex1[v] - ex0[v]) * p.idz_, dxEz = (ezp - ez[v]) * p.idx_;
          const T dxEy = (eyp - ey0[v]) * p.idx_,    dyEx = (exj0[v] - ex0[v]) * p.idy_;
          ax[v] = dyEz * iky_H - dzEy * ikz;
          ay[v] = dzEx * ikz;
          az[v] = -dyEx * iky_H;
          if (!xs) { ay[v] -= dxEz; az[v] += dxEy; }
          else {
            const int si = slab_coord(i0 + v, p.lo[0], p.hi[0], p.nx);
            T ikx = T(1), pyx = T(0), pzx = T(0);
            if (si >= 0 && i0 + v < p.nx && live) {
              ikx = p.kH[0][si];
              const long long q = si + (long long)Sx * (j + (long long)p.ny * k);
              const T b = p.bH[0][si], c = p.cH[0][si];
              pyx = b * fp.psiH_src[pHyx][q] + c * dxEz;
              pzx = b * fp.psiH_src[pHzx][q] + c * dxEy;
              if (owned && it >= 2) { p.psi[pHyx][q] = pyx; p.psi[pHzx][q] = pzx; }
            }
            ay[v] -= dxEz * ikx + pyx;
            az[v] += dxEy * ikx + pzx;
          }
          d0[v] = dyEz; d1[v] = dyEx; d2[v] = dzEy; d3[v] = dzEx;
        }
        if (sj >= 0 && live) {  // y slab: psiHxy (from D+y Ez), psiHzy (from D+y Ex)
          const long long q = i0 + (long long)p.P * (sj + (long long)Sy * k);
          T a[V], d[V];
          ldv(fp.psiH_src[pHxy] + q, a); ldv(fp.psiH_src[pHzy] + q, d);
#pragma unroll
          for (int v = 0; v < V; ++v) {
            a[v] = bHy * a[v] + cHy * d0[v]; d[v] = bHy * d[v] + cHy * d1[v];
            if (i0 + v >= p.nx) { a[v] = T(0); d[v] = T(0); }
            ax[v] += a[v]; az[v] -= d[v];
          }
          if (owned && it >= 2) { stv(p.psi[pHxy] + q, a); stv(p.psi[pHzy] + q, d); }
        }
        if (sk >= 0 && live) {  // z slab: psiHxz (from D+z Ey), psiHyz (from D+z Ex)
          const long long q = i0 + (long long)p.P * (j + (long long)p.ny * sk);
          const T b = p.bH[2][sk], c = p.cH[2][sk];
          T a[V], d[V];
          ldv(fp.psiH_src[pHxz] + q, a); ldv(fp.psiH_src[pHyz] + q, d);
#pragma unroll
          for (int v = 0; v < V; ++v) {
            a[v] = b * a[v] + c * d2[v]; d[v] = b * d[v] + c * d3[v];
            if (i0 + v >= p.nx) { a[v] = T(0); d[v] = T(0); }
            ax[v] -= a[v]; ay[v] += d[v];
          }
          if (owned && it >= 2) { stv(p.psi[pHxz] + q, a); stv(p.psi[pHyz] + q, d); }
        }
        T dbx[V], dby[V], dbz[V];
        if (kMu) {
#pragma unroll
          for (int v = 0; v < V; ++v) { dbx[v] = dby[v] = dbz[v] = T(0); }
          if (live) {
            if (kFull) { ldv(p.Db[0] + o, dbx); ldv(p.Db[1] + o, dby); ldv(p.Db[2] + o, dbz); }
            else {
              unsigned char m[V];
              ld_index<V>(p.idx + o, m);
#pragma unroll
              for (int v = 0; v < V; ++v) {
                dbx[v] = tab[kTabH + 4 * (int)m[v]]; dby[v] = tab[kTabH + 4 * (int)m[v] + 1]; dbz[v] = tab[kTabH + 4 * (int)m[v] + 2];
              }
            }
          }
        } else {
#pragma unroll
          for (int v = 0; v < V; ++v) { dbx[v] = p.db0; dby[v] = p.db0; dbz[v] = p.db0; }
        }
#pragma unroll
        for (int v = 0; v < V; ++v) {
          hx[v] -= dbx[v] * ax[v]; hy[v] -= dby[v] * ay[v]; hz[v] -= dbz[v] * az[v];
          if (!live || i0 + v >= p.nx) { hx[v] = T(0); hy[v] = T(0); hz[v] = T(0); }
        }
        stv(hnb + w * TX + lane * V, hx);
        stv(hnb + (C::ROWS_H + w) * TX + lane * V, hz);
        if (owned && it >= 2) {
          stv_stream(p.dst[kHx] + o, hx); stv_stream(p.dst[kHy] + o, hy); stv_stream(p.dst[kHz] + o, hz);
        }
      }
      // carry the k+1 operands (E^n own values of plane k are still needed by the E phase below: rotate after it)
      if (it >= 2 && w >= 1) {
        // ---------------- sync, then E phase -------------------------------------------------------------------------
        __syncthreads();
        T hxj[V], hzj[V];
        ldv(hnb + (w - 1) * TX + lane * V, hxj);
        ldv(hnb + (C::ROWS_H + w - 1) * TX + lane * V, hzj);
        T hyi = __shfl_up_sync(0xffffffffu, hy[V - 1], 1), hzi = __shfl_up_sync(0xffffffffu, hz[V - 1], 1);
        if (lane == 0) { hyi = hcb[w - 1]; hzi = hcb[TY + w - 1]; }
        const T ikz = sk >= 0 ? p.kE[2][sk] : T(1);
        T ax[V], ay[V], az[V], d0[V], d1[V], d2[V], d3[V];
#pragma unroll
        for (int v = 0; v < V; ++v) {
          const T hym_ = (v > 0) ? hy[v - 1] : hyi;
          const T hzm_ = (v > 0) ? hz[v - 1] : hzi;
          const T dyHz = (hz[v] - hzj[v]) * p.idy_, dzHy = (hy[v] - hym[v]) * p.idz_;
          const T dzHx = (hx[v] - hxm[v]) * p.idz_, dxHz = (hz[v] - hzm_) * p.idx_;
          const T dxHy = (hy[v] - hym_) * p.idx_,   dyHx = (hx[v] - hxj[v]) * p.idy_;
          ax[v] = dyHz * iky_E - dzHy * ikz;
          ay[v] = dzHx * ikz;
          az[v] = -dyHx * iky_E;
          if (!xs) { ay[v] -= dxHz; az[v] += dxHy; }
          else {
            const int si = slab_coord(i0 + v, p.lo[0], p.hi[0], p.nx);
            T ikx = T(1), pyx = T(0), pzx = T(0);
            if (si >= 0 && i0 + v < p.nx && owned) {
              ikx = p.kE[0][si];
              const long long q = si + (long long)Sx * (j + (long long)p.ny * k);
              const T b = p.bE[0][si], c = p.cE[0][si];
              pyx = b * p.psi[pEyx][q] + c * dxHz; p.psi[pEyx][q] = pyx;
              pzx = b * p.psi[pEzx][q] + c * dxHy; p.psi[pEzx][q] = pzx;
            }
            ay[v] -= dxHz * ikx + pyx;
            az[v] += dxHy * ikx + pzx;
          }
          d0[v] = dyHz; d1[v] = dyHx; d2[v] = dzHy; d3[v] = dzHx;
        }
        if (owned) {
          if (sj >= 0) {  // y slab: psiExy (from D-y Hz), psiEzy (from D-y Hx)
            const long long q = i0 + (long long)p.P * (sj + (long long)Sy * k);
            T a[V], d[V];
            ldv(p.psi[pExy] + q, a); ldv(p.psi[pEzy] + q, d);
#pragma unroll
            for (int v = 0; v < V; ++v) {
              a[v] = bEy * a[v] + cEy * d0[v]; d[v] = bEy * d[v] + cEy * d1[v];
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
          if (kFull) {
            ldv(p.Ca[0] + o, cax); ldv(p.Ca[1] + o, cay); ldv(p.Ca[2] + o, caz);
            ldv(p.Cb[0] + o, cbx); ldv(p.Cb[1] + o, cby); ldv(p.Cb[2] + o, cbz);
          } else {
#pragma unroll
            for (int v = 0; v < V; ++v) {
              const Vec4<T> a = lds4(tab + 8 * (int)mi[v]), b = lds4(tab + 8 * (int)mi[v] + 4);
              cax[v] = a.a; cay[v] = a.b; caz[v] = a.c; cbx[v] = a.d; cby[v] = b.a; cbz[v] = b.b;
            }
          }
          const bool wj = (j == 0), wk = (k == 0);
          T ex[V], ey[V];
#pragma unroll
          for (int v = 0; v < V; ++v) {
            const bool wi = (i0 + v == 0), pad = (i0 + v >= p.nx);
            ex[v] = cax[v] * ex0[v] + cbx[v] * ax[v];
            ey[v] = cay[v] * ey0[v] + cby[v] * ay[v];
            ez[v] = caz[v] * ez[v] + cbz[v] * az[v];
            if (wj || wk || pad) ex[v] = T(0);
            if (wi || wk || pad) ey[v] = T(0);
            if (wi || wj || pad) ez[v] = T(0);
          }
          stv_stream(p.dst[kEx] + o, ex); stv_stream(p.dst[kEy] + o, ey); stv_stream(p.dst[kEz] + o, ez);
        }
      } else {
        __syncthreads();
        if (threadIdx.x == 0 && it + NS < nIt) issue(it + NS);
      }
#pragma unroll
      for (int v = 0; v < V; ++v) { ex0[v] = ex1[v]; ey0[v] = ey1[v]; exj0[v] = exj1[v]; }
      eyi0 = eyi1;
      if (it >= 1) {
#pragma unroll
        for (int v = 0; v < V; ++v) { hxm[v] = hx[v]; hym[v] = hy[v]; }
      }
    } else {
      // ---------------- H phase, halo column warp: Hy, Hz at (x0-1, y0+lane, k) ---------------------------------------
      const int r = (lane < TY ? lane : 0) + 1;
      const T c_ex1 = sEx[r * BX + V - 1], c_exj1 = sEx[(r + 1) * BX + V - 1];
      const T c_ey1 = sEy[r * BX + V - 1], c_eyp1 = sEy[r * BX + V];
      if (it >= 1) {
        T hyc = T(0), hzc = T(0);
        if (cin && kin) {
          const T ezc = sEz[r * BX + V - 1], ezp = sEz[r * BX + V];
          hyc = sHy[r * BX + V - 1]; hzc = sHz[r * BX + V - 1];
          const T dzEx = (c_ex1 - c_ex0) * p.idz_, dxEz = (ezp - ezc) * p.idx_;
          const T dxEy = (c_eyp0 - c_ey0) * p.idx_, dyEx = (c_exj0 - c_ex0) * p.idy_;
          const int si = slab_coord(i0, p.lo[0], p.hi[0], p.nx);
          T ay = dzEx * (sk >= 0 ? p.kH[2][sk] : T(1));
          T az = -dyEx * iky_H;
          if (si >= 0) {
            const long long q = si + (long long)Sx * (j + (long long)p.ny * k);
            const T b = p.bH[0][si], c = p.cH[0][si], ikx = p.kH[0][si];
            ay -= dxEz * ikx + (b * fp.psiH_src[pHyx][q] + c * dxEz);
            az += dxEy * ikx + (b * fp.psiH_src[pHzx][q] + c * dxEy);
          } else { ay -= dxEz; az += dxEy; }
          if (sj >= 0) az -= bHy * fp.psiH_src[pHzy][i0 + (long long)p.P * (sj + (long long)Sy * k)] + cHy * dyEx;
          if (sk >= 0) ay += p.bH[2][sk] * fp.psiH_src[pHyz][i0 + (long long)p.P * (j + (long long)p.ny * sk)] + p.cH[2][sk] * dzEx;
          T dby = p.db0, dbz = p.db0;
          if (kMu) {
            if (kFull) { dby = p.Db[1][o]; dbz = p.Db[2][o]; }
            else { const int m = p.idx[o]; dby = tab[kTabH + 4 * m + 1]; dbz = tab[kTabH + 4 * m + 2]; }
          }
          hyc -= dby * ay; hzc -= dbz * az;
        }
        if (lane < TY) { hcb[lane] = hyc; hcb[TY + lane] = hzc; }
      }
      __syncthreads();
      c_ex0 = c_ex1; c_exj0 = c_exj1; c_ey0 = c_ey1; c_eyp0 = c_eyp1;
    }
  }
}

}  // namespace fdtd_b200
