// fdtd_step2.cuh -- TWO full leapfrog steps per pass over a box of cells (temporal blocking over E,H,E,H).
//
// Why: the fused step (fdtd_fused.cuh) already moves what one step must move (49 B per cell-update, fp32 indexed) at 0.93 of
// the rate a copy reaches; the only lever left on Mcell-updates/s is the byte count.  Advancing two steps per pass reads
// every field once and writes it once per TWO cell-updates: 24.5 B per cell-update.
//
// What it computes, for every cell c of the box [bx0,bx1) x [by0,by1) x [bz0,bz1):
//     H^{n+1/2} = H^{n-1/2} - Db curl E^n          (H1)      E^{n+1} = Ca E^n     + Cb curl H^{n+1/2}   (E1)
//     H^{n+3/2} = H^{n+1/2} - Db curl E^{n+1}      (H2)      E^{n+2} = Ca E^{n+1} + Cb curl H^{n+3/2}   (E2)
// R5 steps 1-2 twice, plain Yee arithmetic: the box must keep two cells' distance from every CPML cell (nothing inside the
// dependency cone of the box then carries a psi term); the host plan (fdtd_api.cu) advances what is outside the box -- the
// CPML shell -- step by step with the one-step kernels, and the intermediate fields of the box never reach HBM.
// Ports inside the box: the soft source of the first step (R5 step 3: E_z += A g((n+1) dt) between E1 and H2) is added by
// this kernel to E1 on every source sample it computes, as owner or as halo -- the same value k_source adds, by the same
// expression; the source of the second step and its probes run after the kernel on the stored E2, H2.  The probes of the
// first step need E1, H1 on the port planes, which never leave the chip: the host plan recomputes them on a thin band of
// cells around each port plane with the one-step kernels (fdtd_api.cu, enqueue_pair).
//
// How: like the fused step, a block marches along z over a chunk of planes of an (x,y) tile with TMA-staged input planes,
// one warp per tile row.  Instead of special halo warps, every row warp computes all four half steps on the full 32-lane
// row and the region of VALID results shrinks by one cell per half step on the side the stencil reaches to:
//     H1 valid on the whole computed region (inputs carry a +1 halo row / vector),   E1 valid for r >= 1, c >= 1,
//     H2 valid for 1 <= r <= R-2, 1 <= c <= 126,                                  E2 valid for 2 <= r <= R-2, 2 <= c <= 126.
// A tile of R computed rows x 32 lanes therefore OWNS rows 2..R-2 and lanes 1..30 (vector granularity): (R-3) x 30 V cells.
// In z the same cone costs three priming planes per chunk.  Hand-over between neighbouring rows goes through three
// shared-memory buffers (new Hx,Hz of H1; new Ex,Ez of E1; new Hx,Hz of H2), two slots each (plane parity), with one
// mbarrier per (slot, row); x neighbours come from warp shuffles; the planes k-1 a row needs are carried in registers.
// Two slots are enough because a row cannot start plane k+2 before the row above has finished plane k: its H2 waits for
// that row's E1 of the plane before (row 0, which computes no H2, takes the same wait for that reason alone).  The shared
// memory this leaves holds a fourth TMA stage (C3: 4.36 -> 4.27 ms per step of the box).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include <type_traits>

#include "fdtd_fused.cuh"
#include "fdtd_kernels.cuh"
#include "fdtd_params.h"

namespace fdtd_b200 {

constexpr int kStep2MaxSrc = 4;   // driving ports per handle the two-step kernel carries in its parameters

template <typename T>
struct Step2Params {
  CUtensorMap tm[7];     // boxes of the set being read: Ex Ey Ez Hx Hy Hz, then the uint8 material index
  StepParams<T> sp;      // src = set read (time n), dst = set written (time n+2)
  int kz;                // owned planes per z chunk
  int ntx, nty, group;   // tiles in x, y and dispatch group (as in FusedParams)
  int bx0, bx1, by0, by1, bz0, bz1;   // the box; bx0, bx1 multiples of the vector length
  // soft sources whose samples the kernel may compute (any port with a source: the test is per cell).  The device step
  // counter already stands at n + 2 when the kernel runs (the host plan bumps it before): E1 is at time (counter - 1) dt.
  int nsrc;
  struct Src { int is, sj0, sj1, sk0, sk1, waveform; double amp, t0, sigma, f0; } src[kStep2MaxSrc];
  double dt;
};

template <typename T, int R_, int NS_>
struct Step2Cfg {
  static constexpr int V = VecOf<T>::V, TX = 32 * V, R = R_, NS = NS_;
  static constexpr int TYO = R - 3, TXO = TX - 2 * V;   // owned rows, owned cells per row
  // box of field f: width (elements), rows; every box starts at (ox - V, oy - 2)
  __host__ __device__ static constexpr int xw(int f) { return (f == kEy || f == kEz) ? TX + V : TX; }
  __host__ __device__ static constexpr int nr(int f) { return (f == kEx || f == kEz) ? R + 1 : R; }
  __host__ __device__ static constexpr int tx_bytes(int f) { return nr(f) * xw(f) * (int)sizeof(T); }
  __host__ __device__ static constexpr int off(int f) { return f == 0 ? 0 : off(f - 1) + round128(tx_bytes(f - 1)); }
  // (the uint8 material index does not come through TMA here: a box that starts V cells left of a tile would start at a
  // byte address that is not a multiple of 16, which the TMA unit refuses; each thread loads its V index bytes itself)
  static constexpr int STAGE = off(6);
  static constexpr int XSLOT = 2 * R * TX * (int)sizeof(T);   // one hand-over slot: [2 fields][R rows][TX]
  static constexpr int TAB_B = kTabH * (int)sizeof(T);
  static constexpr int NX = 2, NBAR = 2 * NS + 3 * NX * R;
  static constexpr int BAR_B = round128(NBAR * 8);
  static constexpr int O_X1 = NS * STAGE, O_XE = O_X1 + NX * XSLOT, O_X2 = O_XE + NX * XSLOT, O_TAB = O_X2 + NX * XSLOT,
                       O_BAR = O_TAB + TAB_B;
  static constexpr int SMEM = O_BAR + BAR_B;
  static constexpr int THREADS = (R + 1) * 32;
};

// the V material indices of a thread's cells as one packed word (byte v = cell v)
template <int V> __device__ __forceinline__ unsigned ld_index_packed(const uint8_t* p);
template <> __device__ __forceinline__ unsigned ld_index_packed<4>(const uint8_t* p) { return __ldg(reinterpret_cast<const unsigned*>(p)); }
template <> __device__ __forceinline__ unsigned ld_index_packed<2>(const uint8_t* p) { return (unsigned)__ldg(reinterpret_cast<const unsigned short*>(p)); }

template <typename T, int MODE, int R, int NS>
__global__ void __launch_bounds__((R + 1) * 32, 1) k_step2(const __grid_constant__ Step2Params<T> fp) {
  using C = Step2Cfg<T, R, NS>;
  using O = VOps<T, C::V>;
  constexpr int V = C::V, TX = C::TX;
  constexpr int WEx = C::xw(kEx), WEy = C::xw(kEy), WEz = C::xw(kEz);
  constexpr bool kFull = (MODE & kModeFull) != 0, kMu = (MODE & kModeMu) != 0;
  extern __shared__ __align__(1024) unsigned char smem[];
  T* const x1 = reinterpret_cast<T*>(smem + C::O_X1);     // H1: [slot][Hx|Hz][row][TX]
  T* const xe = reinterpret_cast<T*>(smem + C::O_XE);     // E1: [slot][Ex|Ez][row][TX]
  T* const x2 = reinterpret_cast<T*>(smem + C::O_X2);     // H2: [slot][Hx|Hz][row][TX]
  T* const tab = reinterpret_cast<T*>(smem + C::O_TAB);
  uint64_t* const full = reinterpret_cast<uint64_t*>(smem + C::O_BAR);
  uint64_t* const empty = full + NS;
  uint64_t* const rdy1 = full + 2 * NS;            // [NS][R] H1 row in x1
  uint64_t* const rdyE = rdy1 + C::NX * R;            // [NS][R] E1 row in xe
  uint64_t* const rdy2 = rdyE + C::NX * R;            // [NS][R] H2 row in x2
  constexpr int XS = C::XSLOT / (int)sizeof(T);

  const StepParams<T>& p = fp.sp;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  int tile, chunk;
  {
    const int tiles = fp.ntx * fp.nty, nchunk = (fp.bz1 - fp.bz0 + fp.kz - 1) / fp.kz;
    const int per_group = fp.group * nchunk, g = blockIdx.x / per_group;
    const int gsize = min(fp.group, tiles - g * fp.group), rem = blockIdx.x - g * per_group;
    chunk = rem / gsize;
    tile = g * fp.group + (rem - chunk * gsize);
  }
  const int ty_ = tile / fp.ntx;
  const int ox = fp.bx0 + (tile - ty_ * fp.ntx) * C::TXO, oy = fp.by0 + ty_ * C::TYO;   // first owned cell of the tile
  const int k0 = fp.bz0 + chunk * fp.kz, k1 = min(k0 + fp.kz, fp.bz1);
  const int nIt = k1 - k0 + 4;   // it = 0: Ex, Ey of plane k0-2 only; it >= 1: plane k = k0 - 3 + it

  auto issue = [&](int it, int s) {
    const int k = k0 - 3 + it;
    unsigned char* st = smem + s * C::STAGE;
    const unsigned bytes = it == 0 ? (unsigned)(C::tx_bytes(kEx) + C::tx_bytes(kEy))
                                   : (unsigned)(C::tx_bytes(kEx) + C::tx_bytes(kEy) + C::tx_bytes(kEz) + C::tx_bytes(kHx) +
                                                C::tx_bytes(kHy) + C::tx_bytes(kHz));
    mbar_expect_tx(&full[s], bytes);
    tma_load_3d(st + C::off(kEx), &fp.tm[kEx], &full[s], ox - V, oy - 2, k + 2);
    tma_load_3d(st + C::off(kEy), &fp.tm[kEy], &full[s], ox - V, oy - 2, k + 2);
    if (it >= 1) {
      tma_load_3d(st + C::off(kEz), &fp.tm[kEz], &full[s], ox - V, oy - 2, k + 1);
      tma_load_3d(st + C::off(kHx), &fp.tm[kHx], &full[s], ox - V, oy - 2, k + 1);
      tma_load_3d(st + C::off(kHy), &fp.tm[kHy], &full[s], ox - V, oy - 2, k + 1);
      tma_load_3d(st + C::off(kHz), &fp.tm[kHz], &full[s], ox - V, oy - 2, k + 1);
    }
  };

  if (threadIdx.x == 0) {
    for (int s = 0; s < NS; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], R);
    }
    for (int s = 0; s < C::NX; ++s)
      for (int r = 0; r < R; ++r) { mbar_init(&rdy1[s * R + r], 1); mbar_init(&rdyE[s * R + r], 1); mbar_init(&rdy2[s * R + r], 1); }
    mbar_fence_init();
    for (int it = 0; it < NS && it < nIt; ++it) issue(it, it);
  }
  if (!kFull) {
    constexpr int W4 = 16 / (int)sizeof(T);
    const float4* src = reinterpret_cast<const float4*>(p.tab);
    float4* dst = reinterpret_cast<float4*>(tab);
    for (int q = threadIdx.x; q < kTabH / W4; q += C::THREADS) dst[q] = __ldg(src + q);
  }
  __syncthreads();

  if (w == 0) {
    // ================= warp 0: the TMA producer ===========================================================================
    for (int n = NS; n < nIt; ++n) {
      if (lane == 0) {
        const int s = n % NS;
        mbar_wait(&empty[s], ((n / NS) - 1) & 1);   // every row warp is done with what the slot held
        issue(n, s);
      }
      __syncwarp();
    }
    return;
  }

  // ================= warps 1..R: row r of the computed region, j = oy - 2 + r ================================================
  const int r = w - 1;
  const int j = oy - 2 + r, i0 = ox - V + lane * V;
  const bool jin = j >= 0 && j < p.ny;
  const bool rowB = r >= 1 && r <= R - 2;          // rows that compute H2
  const bool rowE2 = r >= 2 && r <= R - 2;         // rows that compute E2 (= the owned rows)
  const bool own_xy = rowE2 && lane >= 1 && lane <= 30 && j < fp.by1 && i0 < fp.bx1;
  const bool wj = (j == 0);
  const T cx = p.db0 * p.idx_, cy = p.db0 * p.idy_, cz = p.db0 * p.idz_;
  const long long orow = (long long)i0 + (long long)p.P * j;
  // per-cell masks of the vector: inside the grid in x (wall column i = 0 handled separately)
  bool xin[V];
#pragma unroll
  for (int v = 0; v < V; ++v) xin[v] = (i0 + v >= 0) && (i0 + v < p.nx);
  const bool clean_xy = j >= 1 && j < p.ny && i0 >= 1 && i0 + V <= p.nx;   // no wall row / column, no cell outside the grid
  // sources with a sample in this thread's cells (bit q = fp.src[q]); the plane range is tested per iteration
  unsigned srcmask = 0;
  for (int q = 0; q < fp.nsrc; ++q)
    if (j >= fp.src[q].sj0 && j <= fp.src[q].sj1 && fp.src[q].is >= i0 && fp.src[q].is < i0 + V) srcmask |= 1u << q;

  const int oEx = r * WEx + lane * V, oEy = r * WEy + lane * V, oEz = r * WEz + lane * V, oH = r * TX + lane * V;

  // registers carried from one plane to the next
  T ex0[V], ey0[V], exj0[V];      // E^n of plane k: Ex(r), Ey(r), Ex(r+1)
  T eyi0 = T(0);                  // Ey^n(k) of the cell right of the vector
  T h1x[V], h1y[V], h1z[V];       // H1 of plane k-1 (own cells)
  T e1x[V], e1y[V], e1z[V];       // E1 of plane k-1
  T h2xm[V], h2ym[V];             // H2 of plane k-2
  unsigned char mip[V];           // material index of plane k-1
  unsigned mw_next = 0;           // packed material index of plane k+1, in flight
#pragma unroll
  for (int v = 0; v < V; ++v) {
    ex0[v] = ey0[v] = exj0[v] = h1x[v] = h1y[v] = h1z[v] = e1x[v] = e1y[v] = e1z[v] = h2xm[v] = h2ym[v] = T(0);
    mip[v] = 0;
  }

  // E = Ca E_old + Cb curl with the material of (plane offset o, index m), then walls / outside-the-grid -> 0
  auto e_update = [&](T (&ex)[V], T (&ey)[V], T (&ez)[V], const T (&ax)[V], const T (&ay)[V], const T (&az)[V],
                      const unsigned char (&m)[V], long long o, int k) {
    if (kFull) {
      // rows / columns / planes outside the grid (the halo of the computed region) have no coefficient cells: nothing is loaded
      // there and the mask below zeroes the result (same test as load_db)
      if (jin && k >= 0 && k < p.nz && i0 >= 0 && i0 < p.nx) {
      T ca[V], cb[V];
      ldv(p.Ca[0] + o, ca); ldv(p.Cb[0] + o, cb);
#pragma unroll
      for (int v = 0; v < V; ++v) ex[v] = fma(cb[v], ax[v], ca[v] * ex[v]);
      ldv(p.Ca[1] + o, ca); ldv(p.Cb[1] + o, cb);
#pragma unroll
      for (int v = 0; v < V; ++v) ey[v] = fma(cb[v], ay[v], ca[v] * ey[v]);
      ldv(p.Ca[2] + o, ca); ldv(p.Cb[2] + o, cb);
#pragma unroll
      for (int v = 0; v < V; ++v) ez[v] = fma(cb[v], az[v], ca[v] * ez[v]);
      }
    } else {
#pragma unroll
      for (int v = 0; v < V; ++v) {   // (one look-up for vectors under a single material measured slower: 5.21 against 4.80 ms)
        const Vec4<T> a = lds4(tab + 8 * (int)m[v]), b = lds4(tab + 8 * (int)m[v] + 4);
        ex[v] = fma(a.d, ax[v], a.a * ex[v]);
        ey[v] = fma(b.a, ay[v], a.b * ey[v]);
        ez[v] = fma(b.b, az[v], a.c * ez[v]);
      }
    }
    // walls and cells outside the grid -> 0; vectors wholly inside the grid and off the wall rows / columns / plane skip this
    if (!(clean_xy && k >= 1 && k < p.nz)) {
      const bool kin = k >= 0 && k < p.nz, wk = (k == 0) && !p.z_lo_open;
#pragma unroll
      for (int v = 0; v < V; ++v) {
        const bool in = jin && kin && xin[v], wi = (i0 + v == 0);
        if (!in || wj || wk) ex[v] = T(0);
        if (!in || wi || wk) ey[v] = T(0);
        if (!in || wi || wj) ez[v] = T(0);
      }
    }
  };
  // per-cell Db of plane offset o (permeability given), zero outside the grid
  auto load_db = [&](T (&dbx)[V], T (&dby)[V], T (&dbz)[V], const unsigned char (&m)[V], long long o, int k) {
#pragma unroll
    for (int v = 0; v < V; ++v) { dbx[v] = dby[v] = dbz[v] = T(0); }
    if (jin && k >= 0 && k < p.nz && i0 >= 0 && i0 < p.nx) {
      if (kFull) { ldv(p.Db[0] + o, dbx); ldv(p.Db[1] + o, dby); ldv(p.Db[2] + o, dbz); }
      else {
#pragma unroll
        for (int v = 0; v < V; ++v) {
          const Vec4<T> d = ld4(p.tab + kTabH + 4 * (int)m[v]);
          dbx[v] = d.a; dby[v] = d.b; dbz[v] = d.c;
        }
      }
    }
  };

  int s = 0, sprev = 0;
  unsigned ph = 0, phprev = 0;
  long long o = orow + p.PS * (long long)(k0 - 3);

  // One plane iteration.  ST (steady state) = every half step of this row runs in this iteration: the row owns cells
  // (rowE2) and it >= 4.  The priming iterations and the rows at the rim of the computed region (which skip the half steps
  // their results are not valid for) take the general form, which tests each half step and zero-fills what it skips; the
  // steady form carries no such tests and no fills (36 % of the instructions of the first version of this loop).
  auto plane = [&](auto steady, const int it) {
    constexpr bool ST = decltype(steady)::value;
    const int k = k0 - 3 + it, kb = k - 1;
    const unsigned char* st = smem + s * C::STAGE;
    const T* sEx = reinterpret_cast<const T*>(st + C::off(kEx));
    const T* sEy = reinterpret_cast<const T*>(st + C::off(kEy));
    const T* sEz = reinterpret_cast<const T*>(st + C::off(kEz));
    const T* sHx = reinterpret_cast<const T*>(st + C::off(kHx));
    const T* sHy = reinterpret_cast<const T*>(st + C::off(kHy));
    const T* sHz = reinterpret_cast<const T*>(st + C::off(kHz));
    const int xs = it & 1, xsp = xs ^ 1;
    const unsigned xph = (it >> 1) & 1, xphp = ((it - 1) >> 1) & 1;
    T* const x1b = x1 + xs * XS;
    T* const xeb = xe + xs * XS;
    T* const x2b = x2 + xs * XS;
    const T* const xep = xe + xsp * XS;       // E1 of plane k-1, written during the previous iteration

    // material index of the thread's V cells, as ONE packed word: plane k was requested an iteration ago, plane k + 1 is
    // requested now and stays packed until its use (unpacking at once makes the thread wait for the load right here:
    // 20 % of the stall samples of the first version)
    const unsigned mw = mw_next;
    mw_next = 0;
    if (!kFull && jin && k + 1 >= 0 && k + 1 < p.nz && i0 >= 0 && i0 < p.nx) mw_next = ld_index_packed<V>(p.idx + o + p.PS);
    unsigned char mi[V];

    mbar_wait(&full[s], ph);
    T ex1[V], ey1[V], exj1[V];                   // E^n of plane k+1
    ldv(sEx + oEx, ex1); ldv(sEy + oEy, ey1); ldv(sEx + oEx + WEx, exj1);
    T eyi1 = __shfl_down_sync(0xffffffffu, ey1[0], 1);
    if (lane == 31) eyi1 = sEy[oEy + V];
    T hx[V], hy[V], hz[V], ez[V];
    T nex[V], ney[V], nez[V];                    // E1 of plane k
    if (!ST) {
#pragma unroll
      for (int v = 0; v < V; ++v) { hx[v] = hy[v] = hz[v] = ez[v] = nex[v] = ney[v] = nez[v] = T(0); mi[v] = 0; }
    }
    if (ST || it >= 1) {
      // ---------------- H1(k) = H^{n-1/2}(k) - Db curl E^n ------------------------------------------------------------------
      T ezj[V];
      ldv(sEz + oEz, ez); ldv(sEz + oEz + WEz, ezj);
      T ezi = __shfl_down_sync(0xffffffffu, ez[0], 1);
      if (lane == 31) ezi = sEz[oEz + V];
      ldv(sHx + oH, hx); ldv(sHy + oH, hy); ldv(sHz + oH, hz);
      if (kMu && !kFull) {   // per-entry Db: the index is needed already here
#pragma unroll
        for (int v = 0; v < V; ++v) mi[v] = (unsigned char)((mw >> (8 * v)) & 0xffu);
      }
      T dEz_y[V], dEy_z[V], dEx_z[V], dEx_y[V], dEz_x[V], dEy_x[V];
      O::sub(dEz_y, ezj, ez); O::sub(dEy_z, ey1, ey0); O::sub(dEx_z, ex1, ex0); O::sub(dEx_y, exj0, ex0);
#pragma unroll
      for (int v = 0; v < V; ++v) {
        dEz_x[v] = ((v + 1 < V) ? ez[v + 1] : ezi) - ez[v];
        dEy_x[v] = ((v + 1 < V) ? ey0[v + 1] : eyi0) - ey0[v];
      }
      if (!kMu) {
        O::fma_s(hx, dEz_y, -cy); O::fma_s(hx, dEy_z, cz);
        O::fma_s(hy, dEx_z, -cz); O::fma_s(hy, dEz_x, cx);
        O::fma_s(hz, dEy_x, -cx); O::fma_s(hz, dEx_y, cy);
      } else {
        T dbx[V], dby[V], dbz[V];
        load_db(dbx, dby, dbz, mi, o, k);
#pragma unroll
        for (int v = 0; v < V; ++v) {
          hx[v] -= dbx[v] * (dEz_y[v] * p.idy_ - dEy_z[v] * p.idz_);
          hy[v] -= dby[v] * (dEx_z[v] * p.idz_ - dEz_x[v] * p.idx_);
          hz[v] -= dbz[v] * (dEy_x[v] * p.idx_ - dEx_y[v] * p.idy_);
        }
      }
      stv(x1b + oH, hx); stv(x1b + R * TX + oH, hz);
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&rdy1[xs * R + r]);
    if (ST || (it >= 2 && r >= 1)) {
      // ---------------- E1(k) = Ca E^n(k) + Cb curl H1 ----------------------------------------------------------------------
      mbar_wait(&rdy1[xs * R + r - 1], xph);
#pragma unroll
      for (int v = 0; v < V; ++v) mi[v] = (unsigned char)((mw >> (8 * v)) & 0xffu);
      T hxj[V], hzj[V];
      ldv(x1b + oH - TX, hxj); ldv(x1b + R * TX + oH - TX, hzj);
      T hyi = __shfl_up_sync(0xffffffffu, hy[V - 1], 1), hzi = __shfl_up_sync(0xffffffffu, hz[V - 1], 1);
      if (lane == 0) { hyi = T(0); hzi = T(0); }     // c = 0 is outside the valid region of E1 anyway
      T dHz_y[V], dHy_z[V], dHx_z[V], dHx_y[V], dHz_x[V], dHy_x[V];
      O::sub(dHz_y, hz, hzj); O::sub(dHy_z, hy, h1y); O::sub(dHx_z, hx, h1x); O::sub(dHx_y, hx, hxj);
#pragma unroll
      for (int v = 0; v < V; ++v) {
        dHz_x[v] = hz[v] - ((v > 0) ? hz[v - 1] : hzi);
        dHy_x[v] = hy[v] - ((v > 0) ? hy[v - 1] : hyi);
      }
      T ax[V], ay[V], az[V];
      O::mul_s(ax, dHz_y, p.idy_); O::fma_s(ax, dHy_z, -p.idz_);
      O::mul_s(ay, dHx_z, p.idz_); O::fma_s(ay, dHz_x, -p.idx_);
      O::mul_s(az, dHy_x, p.idx_); O::fma_s(az, dHx_y, -p.idy_);
#pragma unroll
      for (int v = 0; v < V; ++v) { nex[v] = ex0[v]; ney[v] = ey0[v]; nez[v] = ez[v]; }
      e_update(nex, ney, nez, ax, ay, az, mi, o, k);
      if (srcmask != 0) {   // R5 step 3 of the first step, in port order (overlapping source boxes add up as k_source adds them)
        const double t = (double)(*p.nstep - 1) * fp.dt;
        for (int q = 0; q < fp.nsrc; ++q) {
          if (!((srcmask >> q) & 1u) || k < fp.src[q].sk0 || k >= fp.src[q].sk1) continue;
          const T g = (T)(fp.src[q].amp * waveform_dev(fp.src[q].waveform, t, fp.src[q].t0, fp.src[q].sigma, fp.src[q].f0));
#pragma unroll
          for (int v = 0; v < V; ++v) if (i0 + v == fp.src[q].is) nez[v] += g;
        }
      }
      stv(xeb + oH, nex); stv(xeb + R * TX + oH, nez);
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&rdyE[xs * R + r]);
    T g2x[V], g2y[V], g2z[V];                    // H2 of plane k-1
    if (!ST) {
#pragma unroll
      for (int v = 0; v < V; ++v) { g2x[v] = g2y[v] = g2z[v] = T(0); }
    }
    if (!ST && r == 0 && it >= 3) mbar_wait(&rdyE[xsp * R + 1], xphp);
    if (ST || (it >= 3 && rowB)) {
      // ---------------- H2(k-1) = H1(k-1) - Db curl E1 ---------------------------------------------------------------------
      mbar_wait(&rdyE[xsp * R + r + 1], xphp);
      T exj[V], ezj[V];
      ldv(xep + oH + TX, exj); ldv(xep + R * TX + oH + TX, ezj);
      T ezi = __shfl_down_sync(0xffffffffu, e1z[0], 1), eyi = __shfl_down_sync(0xffffffffu, e1y[0], 1);
      if (lane == 31) { ezi = T(0); eyi = T(0); }    // c = 127 is outside the valid region of H2 anyway
      T dEz_y[V], dEy_z[V], dEx_z[V], dEx_y[V], dEz_x[V], dEy_x[V];
      O::sub(dEz_y, ezj, e1z); O::sub(dEy_z, ney, e1y); O::sub(dEx_z, nex, e1x); O::sub(dEx_y, exj, e1x);
#pragma unroll
      for (int v = 0; v < V; ++v) {
        dEz_x[v] = ((v + 1 < V) ? e1z[v + 1] : ezi) - e1z[v];
        dEy_x[v] = ((v + 1 < V) ? e1y[v + 1] : eyi) - e1y[v];
        g2x[v] = h1x[v]; g2y[v] = h1y[v]; g2z[v] = h1z[v];
      }
      if (!kMu) {
        O::fma_s(g2x, dEz_y, -cy); O::fma_s(g2x, dEy_z, cz);
        O::fma_s(g2y, dEx_z, -cz); O::fma_s(g2y, dEz_x, cx);
        O::fma_s(g2z, dEy_x, -cx); O::fma_s(g2z, dEx_y, cy);
      } else {
        T dbx[V], dby[V], dbz[V];
        load_db(dbx, dby, dbz, mip, o - p.PS, kb);
#pragma unroll
        for (int v = 0; v < V; ++v) {
          g2x[v] -= dbx[v] * (dEz_y[v] * p.idy_ - dEy_z[v] * p.idz_);
          g2y[v] -= dby[v] * (dEx_z[v] * p.idz_ - dEz_x[v] * p.idx_);
          g2z[v] -= dbz[v] * (dEy_x[v] * p.idx_ - dEx_y[v] * p.idy_);
        }
      }
      stv(x2b + oH, g2x); stv(x2b + R * TX + oH, g2z);
      if (own_xy && (ST || it >= 4)) {
        const long long ob = o - p.PS;
        stv_stream(p.dst[kHx] + ob, g2x); stv_stream(p.dst[kHy] + ob, g2y); stv_stream(p.dst[kHz] + ob, g2z);
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&rdy2[xs * R + r]);
    if (ST || (it >= 4 && rowE2)) {
      // ---------------- E2(k-1) = Ca E1(k-1) + Cb curl H2 -------------------------------------------------------------------
      mbar_wait(&rdy2[xs * R + r - 1], xph);
      T hxj[V], hzj[V];
      ldv(x2b + oH - TX, hxj); ldv(x2b + R * TX + oH - TX, hzj);
      T hyi = __shfl_up_sync(0xffffffffu, g2y[V - 1], 1), hzi = __shfl_up_sync(0xffffffffu, g2z[V - 1], 1);
      if (lane == 0) { hyi = T(0); hzi = T(0); }
      T dHz_y[V], dHy_z[V], dHx_z[V], dHx_y[V], dHz_x[V], dHy_x[V];
      O::sub(dHz_y, g2z, hzj); O::sub(dHy_z, g2y, h2ym); O::sub(dHx_z, g2x, h2xm); O::sub(dHx_y, g2x, hxj);
#pragma unroll
      for (int v = 0; v < V; ++v) {
        dHz_x[v] = g2z[v] - ((v > 0) ? g2z[v - 1] : hzi);
        dHy_x[v] = g2y[v] - ((v > 0) ? g2y[v - 1] : hyi);
      }
      T ax[V], ay[V], az[V];
      O::mul_s(ax, dHz_y, p.idy_); O::fma_s(ax, dHy_z, -p.idz_);
      O::mul_s(ay, dHx_z, p.idz_); O::fma_s(ay, dHz_x, -p.idx_);
      O::mul_s(az, dHy_x, p.idx_); O::fma_s(az, dHx_y, -p.idy_);
      T fx[V], fy[V], fz[V];
#pragma unroll
      for (int v = 0; v < V; ++v) { fx[v] = e1x[v]; fy[v] = e1y[v]; fz[v] = e1z[v]; }
      e_update(fx, fy, fz, ax, ay, az, mip, o - p.PS, kb);
      if (own_xy) {
        const long long ob = o - p.PS;
        stv_stream(p.dst[kEx] + ob, fx); stv_stream(p.dst[kEy] + ob, fy); stv_stream(p.dst[kEz] + ob, fz);
      }
    }
    // release the stage: from here on nothing of this iteration reads it or the hand-over slots of this iteration
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[s]);
    // rotate the carried planes
#pragma unroll
    for (int v = 0; v < V; ++v) {
      ex0[v] = ex1[v]; ey0[v] = ey1[v]; exj0[v] = exj1[v];
      h2xm[v] = g2x[v]; h2ym[v] = g2y[v];
      h1x[v] = hx[v]; h1y[v] = hy[v]; h1z[v] = hz[v];
      e1x[v] = nex[v]; e1y[v] = ney[v]; e1z[v] = nez[v];
      mip[v] = mi[v];
    }
    eyi0 = eyi1;
    sprev = s; phprev = ph;
    if (++s == NS) { s = 0; ph ^= 1u; }
    o += p.PS;
  };

  int it = 0;
  const int n_general = rowE2 ? min(4, nIt) : nIt;
  for (; it < n_general; ++it) plane(std::false_type{}, it);
#pragma unroll 2
  for (; it < nIt; ++it) plane(std::true_type{}, it);
}

}  // namespace fdtd_b200
