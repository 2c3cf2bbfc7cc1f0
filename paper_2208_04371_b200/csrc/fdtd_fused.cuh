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
//     Hx, Hy, Hz of plane k and the uint8 index tile.  Every field has its own box: only the halo it really needs
//     (Hx none in x, Ex/Hy/Hz one vector on the low side, Ey/Ez both sides; Hy no halo row, Ex/Ez two, the rest one),
//     zero-filled outside the array.  NS stages ring with a full and an empty mbarrier per stage.
//   * warp roles, no block-wide barrier anywhere in the plane loop:
//       warp 0         producer: an elected lane re-arms a stage as soon as every consumer warp has released it; the
//                      warp also recomputes Hy, Hz of the halo column i = x0-1 (lane l <-> row y0+l) into shared memory
//       warp 1         halo row j = y0-1: recomputes its Hx, Hz (the j-1 operands of the first owned row)
//       warp 2..TY+1   one owned tile row each: H phase, then E phase
//     New Hx, Hz rows go to a ring of NS shared-memory buffers; row r signals an mbarrier per (buffer, row) and row r+1
//     waits on it before its E phase (point-to-point, so warps drift freely and latencies overlap).  Hy and the k-1
//     plane of Hx, Hy stay in registers; the x-1 operands come from warp shuffles (lane 0: the halo column).
//     A stage is released after the E phase has read the neighbour row, which is also what makes the ring of H buffers
//     safe to overwrite NS planes later.
//   * dispatch order (1-D grid): a group of neighbouring tiles -- as many whole rows of x tiles as fit the SMs -- goes
//     through ALL its z chunks (12..48 planes each) before the next group.  Blocks that run together are then close in z
//     and adjacent in (x,y): their streams stay in a narrow band of the arrays (DRAM locality), halo rows / columns of
//     neighbours and the two priming planes a chunk shares with the tile's previous chunk hit in L2.  Measured on C3: one
//     chunk per tile 13.1 ms, 128-plane chunks 9.0 ms, 12-plane chunks in group order 7.8 ms (profiles/).
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
  int kz;                // planes per z chunk
  int ntx, nty, group;   // tiles in x, y; dispatch order: groups of `group` tiles, all z chunks of a group in ascending
                         // order before the next group (1-D grid: block -> (group, chunk, tile of the group))
  const T* cpack;        // the 18 CPML vectors [axis][bE cE kE bH cH kH][kMaxSlab], contiguous
  T* peer_H[2];          // z slab linked to its upper neighbour (fdtd_z_link): that slab's halo plane -1 of Hx, Hy in the
                         // set this launch writes (element (0,0) of the plane, same pitch); nullptr = not linked
};

__host__ __device__ constexpr int round128(int v) { return (v + 127) / 128 * 128; }

template <typename T, int TY_, int NS_>
struct FusedCfg {
  static constexpr int V = VecOf<T>::V, TX = 32 * V, TY = TY_, NS = NS_;
  // box of field f (Ex Ey Ez Hx Hy Hz): low-side x halo (elements), row width, first row relative to y0, rows
  __host__ __device__ static constexpr int xl(int f) { return f == kHx ? 0 : V; }
  __host__ __device__ static constexpr int xw(int f) { return f == kHx ? TX : ((f == kEy || f == kEz) ? TX + 2 * V : TX + V); }
  __host__ __device__ static constexpr int r0(int f) { return f == kHy ? 0 : -1; }
  __host__ __device__ static constexpr int nr(int f) { return (f == kEx || f == kEz) ? TY + 2 : (f == kHy ? TY : TY + 1); }
  __host__ __device__ static constexpr int tx_bytes(int f) { return nr(f) * xw(f) * (int)sizeof(T); }
  __host__ __device__ static constexpr int off(int f) { return f == 0 ? 0 : off(f - 1) + round128(tx_bytes(f - 1)); }
  static constexpr int I_TX = TY * TX, I_OFF = off(6);
  static constexpr int STAGE = I_OFF + round128(I_TX);
  static constexpr int HN_SLOT = 2 * TY * TX * (int)sizeof(T);          // [Hx|Hz][row 0..TY-1 = j - (y0-1)][x]
  static constexpr int HC_SLOT = round128(2 * TY * (int)sizeof(T));     // [Hy|Hz][row] at i = x0-1
  static constexpr int TAB_B = kTabH * (int)sizeof(T);                  // E records only; Db records are read from global
  static constexpr int CP_B = 3 * 6 * kMaxSlab * (int)sizeof(T);        // CPML vectors [axis][bE cE kE bH cH kH][slab coordinate]
  static constexpr int NBAR = 2 * NS + NS * TY + NS;                    // full, empty, row-ready, column-ready
  static constexpr int BAR_B = round128(NBAR * 8);
  static constexpr int O_HN = NS * STAGE, O_HC = O_HN + NS * HN_SLOT, O_TAB = O_HC + NS * HC_SLOT, O_CP = O_TAB + TAB_B,
                       O_BAR = O_CP + CP_B;
  static constexpr int SMEM = O_BAR + BAR_B;
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
__device__ __forceinline__ void mbar_arrive(uint64_t* b) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
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

// ---- arithmetic on a thread's V consecutive cells; fp32 uses the packed two-wide FP32 pipe (FFMA2) --------------------
template <typename T, int V> struct VOps {
  static __device__ __forceinline__ void sub(T (&r)[V], const T (&a)[V], const T (&b)[V]) {
#pragma unroll
    for (int v = 0; v < V; ++v) r[v] = a[v] - b[v];
  }
  static __device__ __forceinline__ void fma_s(T (&r)[V], const T (&a)[V], T s) {  // r += a * s
#pragma unroll
    for (int v = 0; v < V; ++v) r[v] = fma(a[v], s, r[v]);
  }
  static __device__ __forceinline__ void mul_s(T (&r)[V], const T (&a)[V], T s) {
#pragma unroll
    for (int v = 0; v < V; ++v) r[v] = a[v] * s;
  }
};
template <> struct VOps<float, 4> {
  static __device__ __forceinline__ void sub(float (&r)[4], const float (&a)[4], const float (&b)[4]) {
    const float2 m1 = make_float2(-1.f, -1.f);
    const float2 lo = __ffma2_rn(make_float2(b[0], b[1]), m1, make_float2(a[0], a[1]));
    const float2 hi = __ffma2_rn(make_float2(b[2], b[3]), m1, make_float2(a[2], a[3]));
    r[0] = lo.x; r[1] = lo.y; r[2] = hi.x; r[3] = hi.y;
  }
  static __device__ __forceinline__ void fma_s(float (&r)[4], const float (&a)[4], float s) {
    const float2 ss = make_float2(s, s);
    const float2 lo = __ffma2_rn(make_float2(a[0], a[1]), ss, make_float2(r[0], r[1]));
    const float2 hi = __ffma2_rn(make_float2(a[2], a[3]), ss, make_float2(r[2], r[3]));
    r[0] = lo.x; r[1] = lo.y; r[2] = hi.x; r[3] = hi.y;
  }
  static __device__ __forceinline__ void mul_s(float (&r)[4], const float (&a)[4], float s) {
    const float2 ss = make_float2(s, s);
    const float2 lo = __fmul2_rn(make_float2(a[0], a[1]), ss);
    const float2 hi = __fmul2_rn(make_float2(a[2], a[3]), ss);
    r[0] = lo.x; r[1] = lo.y; r[2] = hi.x; r[3] = hi.y;
  }
};

__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// ------------------------------------------------------------------------------------------------------------------
// k_step_fused.  Structure of one plane iteration (all warps): wait for the stage -> H phase -> __syncthreads -> E phase.
// The arithmetic is written as the plain Yee update (kappa = 1, psi = 0) for every cell, followed by additive CPML
// corrections under warp-uniform (y slab, z slab) or per-lane (x slab) branches:
//     H -= Db * [ (1/kappa - 1) * dE + psi ]        E += Cb * [ (1/kappa - 1) * dH + psi ]
// which is R5 regrouped (identical up to rounding).  Cells outside the grid (halo of edge tiles, pad columns) need no
// masks in the plain H update: all their operands are zeros supplied by TMA / the zero pad, so their results are zeros.
// ------------------------------------------------------------------------------------------------------------------
// psi <- b psi + c d  for a thread's V cells of two psi arrays (cells at or beyond nx stay zero)
template <typename T, int V>
__device__ __forceinline__ void psi_update2(T (&a)[V], T (&d)[V], const T (&da)[V], const T (&dd)[V], T b, T c, T inv, int nvalid) {
#pragma unroll
  for (int v = 0; v < V; ++v) {
    a[v] = b * a[v] + (c * inv) * da[v];
    d[v] = b * d[v] + (c * inv) * dd[v];
    if (v >= nvalid) { a[v] = T(0); d[v] = T(0); }
  }
}

// Tiles of at most kFusedSmallTY rows are the small-tile build: two blocks per SM (their shared memory and 128 registers per
// thread allow it), so that two independent z marches hide each other's latencies on grids whose tiles are mostly CPML
// rows / columns or too few to fill the SMs with one block each (DESIGN.md 6.2 "mid-size grids").
constexpr int kFusedSmallTY = 6;
template <typename T, int MODE, int TY, int NS>
__global__ void __launch_bounds__((TY + 2) * 32, (TY <= kFusedSmallTY ? 2 : 1)) k_step_fused(const __grid_constant__ FusedParams<T> fp) {
  using C = FusedCfg<T, TY, NS>;
  using O = VOps<T, C::V>;
  constexpr int V = C::V, TX = C::TX;
  constexpr int WEx = C::xw(kEx), WEy = C::xw(kEy), WEz = C::xw(kEz), WHy = C::xw(kHy), WHz = C::xw(kHz);
  constexpr bool kFull = (MODE & kModeFull) != 0, kMu = (MODE & kModeMu) != 0;
  extern __shared__ __align__(1024) unsigned char smem[];
  T* const hn = reinterpret_cast<T*>(smem + C::O_HN);
  T* const hc = reinterpret_cast<T*>(smem + C::O_HC);
  T* const tab = reinterpret_cast<T*>(smem + C::O_TAB);
  T* const cpv = reinterpret_cast<T*>(smem + C::O_CP);
  uint64_t* const full = reinterpret_cast<uint64_t*>(smem + C::O_BAR);  // [NS] TMA bytes of the stage have landed
  uint64_t* const empty = full + NS;                                     // [NS] every consumer warp is done with the stage
  uint64_t* const rowrdy = full + 2 * NS;                                // [NS][TY] new Hx, Hz of row r are in hn[slot]
  uint64_t* const colrdy = full + 2 * NS + NS * TY;                      // [NS] halo column Hy, Hz are in hc[slot]
  // CPML vector v (0..5 = bE cE kE bH cH kH) of axis a at slab coordinate q
  auto cp = [&](int a, int v, int q) -> T { return cpv[(a * 6 + v) * kMaxSlab + q]; };

  const StepParams<T>& p = fp.sp;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  // block -> (tile, chunk).  The hardware dispatches blocks in index order, so the co-resident blocks are `group`
  // neighbouring tiles at (nearly) the same chunk: their streams stay within a narrow band of planes, halo rows/columns
  // of neighbours hit in L2, and a tile's next chunk follows one wave after the previous one.
  int tile, chunk;
  {
    const int tiles = fp.ntx * fp.nty, nchunk = (p.nz + fp.kz - 1) / fp.kz;
    const int per_group = fp.group * nchunk, g = blockIdx.x / per_group;
    const int gsize = min(fp.group, tiles - g * fp.group), rem = blockIdx.x - g * per_group;
    chunk = rem / gsize;
    tile = g * fp.group + (rem - chunk * gsize);
  }
  const int ty_ = tile / fp.ntx;
  const int x0 = (tile - ty_ * fp.ntx) * TX, y0 = ty_ * TY;
  const int k0 = chunk * fp.kz, k1 = min(k0 + fp.kz, p.nz);
  const int nIt = k1 - k0 + 2;  // it = 0: Ex, Ey of plane k0-1 only; it = 1: H of plane k0-1; it >= 2: plane k0 + it - 2

  if (blockIdx.x == 0 && threadIdx.x == 0) *p.nstep += 1;

  // one elected thread issues the boxes of iteration `it` (plane k) into stage s
  auto issue = [&](int it, int s) {
    const int k = k0 - 2 + it;
    unsigned char* st = smem + s * C::STAGE;
    const bool want_idx = !kFull && it >= 2;
    // it = 1 (plane k0-1) exists only for its new Hx, Hy (the k-1 operands of plane k0): old Hz is not needed there
    const unsigned bytes = it == 0 ? (unsigned)(C::tx_bytes(kEx) + C::tx_bytes(kEy))
                                   : (unsigned)(C::tx_bytes(kEx) + C::tx_bytes(kEy) + C::tx_bytes(kEz) + C::tx_bytes(kHx) +
                                                C::tx_bytes(kHy)) + (it >= 2 ? (unsigned)C::tx_bytes(kHz) : 0u) +
                                         (want_idx ? (unsigned)C::I_TX : 0u);
    mbar_expect_tx(&full[s], bytes);
    // Ex, Ey: plane k+1 (array plane index + 1); the rest: plane k
    tma_load_3d(st + C::off(kEx), &fp.tm[kEx], &full[s], x0 - C::xl(kEx), y0 + C::r0(kEx), k + 2);
    tma_load_3d(st + C::off(kEy), &fp.tm[kEy], &full[s], x0 - C::xl(kEy), y0 + C::r0(kEy), k + 2);
    if (it >= 1) {
      tma_load_3d(st + C::off(kEz), &fp.tm[kEz], &full[s], x0 - C::xl(kEz), y0 + C::r0(kEz), k + 1);
      tma_load_3d(st + C::off(kHx), &fp.tm[kHx], &full[s], x0 - C::xl(kHx), y0 + C::r0(kHx), k + 1);
      tma_load_3d(st + C::off(kHy), &fp.tm[kHy], &full[s], x0 - C::xl(kHy), y0 + C::r0(kHy), k + 1);
      if (it >= 2) tma_load_3d(st + C::off(kHz), &fp.tm[kHz], &full[s], x0 - C::xl(kHz), y0 + C::r0(kHz), k + 1);
      if (want_idx) tma_load_3d(st + C::I_OFF, &fp.tm[6], &full[s], x0, y0, k + 1);
    }
  };

  if (threadIdx.x == 0) {
    for (int s = 0; s < NS; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], TY + 1);   // warps 1..TY+1
      mbar_init(&colrdy[s], 1);
      for (int r = 0; r < TY; ++r) mbar_init(&rowrdy[s * TY + r], 1);
    }
    mbar_fence_init();
    // the first NS planes are requested before anything else so that their latency overlaps the table copies below
    for (int it = 0; it < NS && it < nIt; ++it) issue(it, it);
  }
  {  // material table (E records) and CPML vectors -> shared memory, 128 bits per thread and round
    constexpr int W4 = 16 / (int)sizeof(T);
    if (!kFull) {
      const float4* src = reinterpret_cast<const float4*>(p.tab);
      float4* dst = reinterpret_cast<float4*>(tab);
      for (int q = threadIdx.x; q < kTabH / W4; q += C::THREADS) dst[q] = __ldg(src + q);
    }
    const float4* src = reinterpret_cast<const float4*>(fp.cpack);
    float4* dst = reinterpret_cast<float4*>(cpv);
    for (int q = threadIdx.x; q < 18 * kMaxSlab / W4; q += C::THREADS) dst[q] = __ldg(src + q);
  }
  __syncthreads();

  // ---- loop invariants ------------------------------------------------------------------------------------------------
  const bool rowwarp = w >= 1;
  const int r = w - 1;  // row warps: tile row index relative to the halo row, j = y0-1+r
  // row warps: j = y0-1+r (r = 0 is the halo row); column warp: lane l <-> row y0+l at i = x0-1
  const int j = rowwarp ? y0 - 1 + r : y0 + lane;
  const int i0 = rowwarp ? x0 + lane * V : x0 - 1;
  const bool jin = j >= 0 && j < p.ny;
  const bool cin = rowwarp ? (jin && i0 < p.nx) : (jin && i0 >= 0 && lane < TY);  // the thread's cell(s) exist
  const bool owned = rowwarp && r >= 1 && cin;                                    // ... and this thread stores them
  const int nvalid = rowwarp ? min(V, p.nx - i0) : 1;                             // cells of the vector inside the grid
  const int Sx = p.Sxp, Sy = p.lo[1] + p.hi[1], Sz = p.lo[2] + p.hi[2];
  const int sj = (cin && Sy > 0) ? slab_coord(j, p.lo[1], p.hi[1], p.ny) : -1;
  // x slab: padded coordinate of the thread's first cell (the x slabs are stored in whole vectors, fdtd_params.h: a row
  // warp's vector is wholly inside or wholly outside, always 128-bit psi accesses)
  const int si0 = (cin && Sx > 0) ? xslab_coord(p, i0) : -1;
  const bool xs = si0 >= 0;
  const bool wj = (j == 0), wi = (i0 == 0);
  const bool xtail = x0 + TX > p.nx;
  const int kzlo = p.lo[2], kzhi = p.nz - p.hi[2];
  // uniform update constants (no permeability arrays): H -= (dt/mu0)/d * dE
  const T cx = p.db0 * p.idx_, cy = p.db0 * p.idy_, cz = p.db0 * p.idz_;
  // psi offsets, evaluated inside the slab branches only (keeps the plain path's register budget small)
  auto qy = [&](int k) { return (long long)i0 + (long long)p.P * (sj + (long long)Sy * k); };              // y slab
  auto qz = [&](int sk) { return (long long)i0 + (long long)p.P * (j + (long long)p.ny * sk); };           // z slab
  auto qx = [&](int k) { return (long long)(si0 >= 0 ? si0 : 0) + (long long)Sx * (j + (long long)p.ny * k); };  // x slab
  const long long orow = (long long)i0 + (long long)p.P * j;

  int s = 0;
  unsigned ph = 0;
  long long o = orow + p.PS * (long long)(k0 - 2);

  if (!rowwarp) {
    // ================= warp 0: halo column Hy, Hz at (x0-1, y0+lane, k), and the TMA producer ==========================
    T c_ex0 = T(0), c_exj0 = T(0), c_ey0 = T(0), c_eyp0 = T(0);  // plane k: Ex(x0-1,j), Ex(x0-1,j+1), Ey(x0-1,j), Ey(x0,j)
    const int rr = lane < TY ? lane : 0;
    for (int it = 0; it < nIt; ++it, o += p.PS) {
      const int k = k0 - 2 + it;
      const unsigned char* st = smem + s * C::STAGE;
      const T* sEx = reinterpret_cast<const T*>(st + C::off(kEx));
      const T* sEy = reinterpret_cast<const T*>(st + C::off(kEy));
      const T* sEz = reinterpret_cast<const T*>(st + C::off(kEz));
      const T* sHy = reinterpret_cast<const T*>(st + C::off(kHy));
      const T* sHz = reinterpret_cast<const T*>(st + C::off(kHz));
      const bool zs = Sz > 0 && k >= 0 && (k < kzlo || k >= kzhi);
      const bool pml = (xs || sj >= 0 || zs) && cin && k >= 0;
      mbar_wait(&full[s], ph);
      const T c_ex1 = sEx[(rr + 1) * WEx + V - 1], c_exj1 = sEx[(rr + 2) * WEx + V - 1];
      const T c_ey1 = sEy[(rr + 1) * WEy + V - 1], c_eyp1 = sEy[(rr + 1) * WEy + V];
      if (it >= 1) {
        const T ezc = sEz[(rr + 1) * WEz + V - 1], ezp = sEz[(rr + 1) * WEz + V];
        T hyc = sHy[rr * WHy + V - 1], hzc = sHz[(rr + 1) * WHz + V - 1];
        const T dEx_z = c_ex1 - c_ex0, dEz_x = ezp - ezc, dEy_x = c_eyp0 - c_ey0, dEx_y = c_exj0 - c_ex0;
        T dby = p.db0, dbz = p.db0;
        if (kMu) {
          dby = dbz = T(0);
          if (cin && k >= 0) {
            if (kFull) { dby = p.Db[1][o]; dbz = p.Db[2][o]; }
            else { const int m = p.idx[o]; dby = p.tab[kTabH + 4 * m + 1]; dbz = p.tab[kTabH + 4 * m + 2]; }
          }
        }
        hyc -= dby * (dEx_z * p.idz_ - dEz_x * p.idx_);
        hzc -= dbz * (dEy_x * p.idx_ - dEx_y * p.idy_);
        if (pml) {
          if (xs) {
            const long long q = qx(k);
            const T b = cp(0, 3, si0), c = cp(0, 4, si0), km1 = cp(0, 5, si0) - T(1);
            const T dz_ = dEz_x * p.idx_, dy_ = dEy_x * p.idx_;
            hyc += dby * (km1 * dz_ + b * fp.psiH_src[pHyx][q] + c * dz_);
            hzc -= dbz * (km1 * dy_ + b * fp.psiH_src[pHzx][q] + c * dy_);
          }
          if (sj >= 0) {
            const T dx_ = dEx_y * p.idy_;
            hzc += dbz * ((cp(1, 5, sj) - T(1)) * dx_ + cp(1, 3, sj) * fp.psiH_src[pHzy][qy(k)] + cp(1, 4, sj) * dx_);
          }
          if (zs) {
            const int sk = slab_coord(k, p.lo[2], p.hi[2], p.nz);
            const T dx_ = dEx_z * p.idz_;
            hyc -= dby * ((cp(2, 5, sk) - T(1)) * dx_ + cp(2, 3, sk) * fp.psiH_src[pHyz][qz(sk)] + cp(2, 4, sk) * dx_);
          }
        }
        T* const hcb = hc + s * (C::HC_SLOT / (int)sizeof(T));
        if (lane < TY) { hcb[lane] = hyc; hcb[TY + lane] = hzc; }
      }
      c_ex0 = c_ex1; c_exj0 = c_exj1; c_ey0 = c_ey1; c_eyp0 = c_eyp1;
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(&colrdy[s]);
        // re-arm the stage of the previous plane once every consumer warp has released it
        if (it >= 1 && it - 1 + NS < nIt) {
          const int ps = s == 0 ? NS - 1 : s - 1;
          mbar_wait(&empty[ps], s == 0 ? ph ^ 1u : ph);
          issue(it - 1 + NS, ps);
        }
      }
      if (++s == NS) { s = 0; ph ^= 1u; }
    }
    return;
  }

  // ================= warps 1..TY+1: row j = y0-1+r ======================================================================
  const int oEx = r * WEx + V + lane * V, oEy = r * WEy + V + lane * V, oEz = r * WEz + V + lane * V;
  const int oHx = r * TX + lane * V, oHy = (r >= 1 ? r - 1 : 0) * WHy + V + lane * V, oHz = r * WHz + V + lane * V;
  const int oHn = r * TX + lane * V;   // own row in the H ring (rows 0..TY-1 are written; row TY has no reader)
  // registers carried from one plane to the next
  T ex0[V], ey0[V], exj0[V], hxm[V], hym[V];
  T eyi0 = T(0);
#pragma unroll
  for (int v = 0; v < V; ++v) { ex0[v] = ey0[v] = exj0[v] = hxm[v] = hym[v] = T(0); }

  for (int it = 0; it < nIt; ++it, o += p.PS) {
    const int k = k0 - 2 + it;
    const unsigned char* st = smem + s * C::STAGE;
    const T* sEx = reinterpret_cast<const T*>(st + C::off(kEx));
    const T* sEy = reinterpret_cast<const T*>(st + C::off(kEy));
    const T* sEz = reinterpret_cast<const T*>(st + C::off(kEz));
    const T* sHx = reinterpret_cast<const T*>(st + C::off(kHx));
    const T* sHy = reinterpret_cast<const T*>(st + C::off(kHy));
    const T* sHz = reinterpret_cast<const T*>(st + C::off(kHz));
    const unsigned char* sIdx = st + C::I_OFF;
    const bool zs = Sz > 0 && k >= 0 && (k < kzlo || k >= kzhi);
    const bool pml = (xs || sj >= 0 || zs) && cin && k >= 0;   // some CPML correction applies to this thread
    T* const hnb = hn + s * (C::HN_SLOT / (int)sizeof(T));

    if (kFull && owned && it >= 1 && it + 1 < nIt) {  // full mode: the next plane's coefficient lines, one plane ahead, into L2
      const long long on = o + p.PS;
#pragma unroll
      for (int c = 0; c < 3; ++c) { prefetch_l2(p.Ca[c] + on); prefetch_l2(p.Cb[c] + on); }
    }
    if (pml && it + 1 < nIt) {  // pull the psi lines of the next plane into L2 while this plane is being processed
      if (sj >= 0) {
        const long long q = qy(k + 1);
        prefetch_l2(fp.psiH_src[pHxy] + q); prefetch_l2(fp.psiH_src[pHzy] + q);
        prefetch_l2(p.psi[pExy] + q); prefetch_l2(p.psi[pEzy] + q);
      }
      if (xs) {
        const long long q = qx(k + 1);
        prefetch_l2(fp.psiH_src[pHyx] + q); prefetch_l2(fp.psiH_src[pHzx] + q);
        prefetch_l2(p.psi[pEyx] + q); prefetch_l2(p.psi[pEzx] + q);
      }
      if (k + 1 < kzlo || k + 1 >= kzhi) {
        if (Sz > 0 && k + 1 >= 0 && k + 1 < p.nz) {
          const long long q = qz(slab_coord(k + 1, p.lo[2], p.hi[2], p.nz));
          prefetch_l2(fp.psiH_src[pHxz] + q); prefetch_l2(fp.psiH_src[pHyz] + q);
          prefetch_l2(p.psi[pExz] + q); prefetch_l2(p.psi[pEyz] + q);
        }
      }
    }

    mbar_wait(&full[s], ph);
    T ex1[V], ey1[V], exj1[V];
    ldv(sEx + oEx, ex1); ldv(sEy + oEy, ey1); ldv(sEx + oEx + WEx, exj1);
    T eyi1 = __shfl_down_sync(0xffffffffu, ey1[0], 1);
    if (lane == 31) eyi1 = sEy[oEy + V];
    T hx[V], hy[V], hz[V], ez[V];
    if (it >= 1) {
      // ---------------- H phase: H^{n+1/2}(k) = H^{n-1/2}(k) - Db curl E^n -------------------------------------------
      T ezj[V];
      ldv(sEz + oEz, ez); ldv(sEz + oEz + WEz, ezj);
      T ezi = __shfl_down_sync(0xffffffffu, ez[0], 1);
      if (lane == 31) ezi = sEz[oEz + V];
      ldv(sHx + oHx, hx); ldv(sHy + oHy, hy); ldv(sHz + oHz, hz);

      T dEz_y[V], dEy_z[V], dEx_z[V], dEx_y[V], dEz_x[V], dEy_x[V];   // undivided differences
      O::sub(dEz_y, ezj, ez); O::sub(dEy_z, ey1, ey0); O::sub(dEx_z, ex1, ex0); O::sub(dEx_y, exj0, ex0);
#pragma unroll
      for (int v = 0; v < V; ++v) {
        dEz_x[v] = ((v + 1 < V) ? ez[v + 1] : ezi) - ez[v];
        dEy_x[v] = ((v + 1 < V) ? ey0[v + 1] : eyi0) - ey0[v];
      }
      T dbx[V], dby[V], dbz[V];
      if (!kMu) {
        O::fma_s(hx, dEz_y, -cy); O::fma_s(hx, dEy_z, cz);
        O::fma_s(hy, dEx_z, -cz); O::fma_s(hy, dEz_x, cx);
        O::fma_s(hz, dEy_x, -cx); O::fma_s(hz, dEx_y, cy);
#pragma unroll
        for (int v = 0; v < V; ++v) { dbx[v] = dby[v] = dbz[v] = p.db0; }
      } else {
#pragma unroll
        for (int v = 0; v < V; ++v) { dbx[v] = dby[v] = dbz[v] = T(0); }
        if (cin && k >= 0) {
          if (kFull) { ldv(p.Db[0] + o, dbx); ldv(p.Db[1] + o, dby); ldv(p.Db[2] + o, dbz); }
          else {
            unsigned char m[V];
            ld_index<V>(p.idx + o, m);
#pragma unroll
            for (int v = 0; v < V; ++v) {
              const Vec4<T> d = ld4(p.tab + kTabH + 4 * (int)m[v]);
              dbx[v] = d.a; dby[v] = d.b; dbz[v] = d.c;
            }
          }
        }
#pragma unroll
        for (int v = 0; v < V; ++v) {
          hx[v] -= dbx[v] * (dEz_y[v] * p.idy_ - dEy_z[v] * p.idz_);
          hy[v] -= dby[v] * (dEx_z[v] * p.idz_ - dEz_x[v] * p.idx_);
          hz[v] -= dbz[v] * (dEy_x[v] * p.idx_ - dEx_y[v] * p.idy_);
        }
      }
      if (pml) {
        const bool wr = owned && it >= 2;
        if (sj >= 0) {  // y slab: psiHxy (from D+y Ez) -> Hx, psiHzy (from D+y Ex) -> Hz
          const long long q = qy(k);
          T a[V], d[V];
          ldv(fp.psiH_src[pHxy] + q, a); ldv(fp.psiH_src[pHzy] + q, d);
          const T ykH = (cp(1, 5, sj) - T(1)) * p.idy_;
          psi_update2<T, V>(a, d, dEz_y, dEx_y, cp(1, 3, sj), cp(1, 4, sj), p.idy_, nvalid);
#pragma unroll
          for (int v = 0; v < V; ++v) {
            hx[v] -= dbx[v] * (ykH * dEz_y[v] + a[v]); hz[v] += dbz[v] * (ykH * dEx_y[v] + d[v]);
          }
          if (wr) { stv(p.psi[pHxy] + q, a); stv(p.psi[pHzy] + q, d); }
        }
        if (zs) {  // z slab: psiHxz (from D+z Ey) -> Hx, psiHyz (from D+z Ex) -> Hy
          const int sk = slab_coord(k, p.lo[2], p.hi[2], p.nz);
          const long long q = qz(sk);
          const T b = cp(2, 3, sk), c = cp(2, 4, sk), km = (cp(2, 5, sk) - T(1)) * p.idz_;
          T a[V], d[V];
          ldv(fp.psiH_src[pHxz] + q, a); ldv(fp.psiH_src[pHyz] + q, d);
          psi_update2<T, V>(a, d, dEy_z, dEx_z, b, c, p.idz_, nvalid);
#pragma unroll
          for (int v = 0; v < V; ++v) {
            hx[v] += dbx[v] * (km * dEy_z[v] + a[v]); hy[v] -= dby[v] * (km * dEx_z[v] + d[v]);
          }
          if (wr) { stv(p.psi[pHxz] + q, a); stv(p.psi[pHyz] + q, d); }
        }
        if (xs) {  // x slab: psiHyx (from D+x Ez) -> Hy, psiHzx (from D+x Ey) -> Hz
          const long long q0 = qx(k);
          T a[V], d[V];
          ldv(fp.psiH_src[pHyx] + q0, a); ldv(fp.psiH_src[pHzx] + q0, d);
#pragma unroll
          for (int v = 0; v < V; ++v) {
            const T b = cp(0, 3, si0 + v), c = cp(0, 4, si0 + v) * p.idx_, km = (cp(0, 5, si0 + v) - T(1)) * p.idx_;
            a[v] = b * a[v] + c * dEz_x[v]; d[v] = b * d[v] + c * dEy_x[v];
            hy[v] += dby[v] * (km * dEz_x[v] + a[v]); hz[v] -= dbz[v] * (km * dEy_x[v] + d[v]);
          }
          if (wr) { stv(p.psi[pHyx] + q0, a); stv(p.psi[pHzx] + q0, d); }
        }
      }
      if (r < TY) { stv(hnb + oHn, hx); stv(hnb + TY * TX + oHn, hz); }
      if (owned && it >= 2) {
        stv_stream(p.dst[kHx] + o, hx); stv_stream(p.dst[kHy] + o, hy); stv_stream(p.dst[kHz] + o, hz);
        // top plane of a linked z slab: the tangential H the slab above needs for its E update on plane 0 goes straight
        // into that slab's halo plane (NVLink peer stores from the kernel that computes them)
        if (k == p.nz - 1 && fp.peer_H[0] != nullptr) { stv(fp.peer_H[0] + orow, hx); stv(fp.peer_H[1] + orow, hy); }
      }
    }
    __syncwarp();
    if (lane == 0 && r < TY) mbar_arrive(&rowrdy[s * TY + r]);   // every iteration, so that the phase parity is it / NS
    if (it >= 2 && r >= 1 && !(p.z_lo_open && k == 0)) {   // plane 0 of a lo-open z slab: E is updated by fdtd_step_end
      // ---------------- E phase: E^{n+1}(k) = Ca E^n + Cb curl H^{n+1/2} ---------------------------------------------
      unsigned char mi[V];
      if (!kFull) ld_index_smem<V>(sIdx + (r - 1) * TX + lane * V, mi);
      mbar_wait(&rowrdy[s * TY + r - 1], ph);
      T hxj[V], hzj[V];
      ldv(hnb + oHn - TX, hxj);
      ldv(hnb + TY * TX + oHn - TX, hzj);
      T hyi = __shfl_up_sync(0xffffffffu, hy[V - 1], 1), hzi = __shfl_up_sync(0xffffffffu, hz[V - 1], 1);
      if (lane == 0) {
        mbar_wait(&colrdy[s], ph);
        const T* const hcb = hc + s * (C::HC_SLOT / (int)sizeof(T));
        hyi = hcb[r - 1]; hzi = hcb[TY + r - 1];
      }
      // release the stage: nothing below reads it or the H ring (the loads above are ordered before the arrive)
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[s]);
      T dHz_y[V], dHy_z[V], dHx_z[V], dHx_y[V], dHz_x[V], dHy_x[V];
      O::sub(dHz_y, hz, hzj); O::sub(dHy_z, hy, hym); O::sub(dHx_z, hx, hxm); O::sub(dHx_y, hx, hxj);
#pragma unroll
      for (int v = 0; v < V; ++v) {
        dHz_x[v] = hz[v] - ((v > 0) ? hz[v - 1] : hzi);
        dHy_x[v] = hy[v] - ((v > 0) ? hy[v - 1] : hyi);
      }
      T ax[V], ay[V], az[V];
      O::mul_s(ax, dHz_y, p.idy_); O::fma_s(ax, dHy_z, -p.idz_);
      O::mul_s(ay, dHx_z, p.idz_); O::fma_s(ay, dHz_x, -p.idx_);
      O::mul_s(az, dHy_x, p.idx_); O::fma_s(az, dHx_y, -p.idy_);
      if (pml && owned) {
        if (sj >= 0) {  // y slab: psiExy (from D-y Hz) -> Ex, psiEzy (from D-y Hx) -> Ez
          const long long q = qy(k);
          T a[V], d[V];
          ldv(p.psi[pExy] + q, a); ldv(p.psi[pEzy] + q, d);
          const T ykE = (cp(1, 2, sj) - T(1)) * p.idy_;
          psi_update2<T, V>(a, d, dHz_y, dHx_y, cp(1, 0, sj), cp(1, 1, sj), p.idy_, nvalid);
#pragma unroll
          for (int v = 0; v < V; ++v) { ax[v] += ykE * dHz_y[v] + a[v]; az[v] -= ykE * dHx_y[v] + d[v]; }
          stv(p.psi[pExy] + q, a); stv(p.psi[pEzy] + q, d);
        }
        if (zs) {  // z slab: psiExz (from D-z Hy) -> Ex, psiEyz (from D-z Hx) -> Ey
          const int sk = slab_coord(k, p.lo[2], p.hi[2], p.nz);
          const long long q = qz(sk);
          const T b = cp(2, 0, sk), c = cp(2, 1, sk), km = (cp(2, 2, sk) - T(1)) * p.idz_;
          T a[V], d[V];
          ldv(p.psi[pExz] + q, a); ldv(p.psi[pEyz] + q, d);
          psi_update2<T, V>(a, d, dHy_z, dHx_z, b, c, p.idz_, nvalid);
#pragma unroll
          for (int v = 0; v < V; ++v) { ax[v] -= km * dHy_z[v] + a[v]; ay[v] += km * dHx_z[v] + d[v]; }
          stv(p.psi[pExz] + q, a); stv(p.psi[pEyz] + q, d);
        }
        if (xs) {  // x slab: psiEyx (from D-x Hz) -> Ey, psiEzx (from D-x Hy) -> Ez
          const long long q0 = qx(k);
          T a[V], d[V];
          ldv(p.psi[pEyx] + q0, a); ldv(p.psi[pEzx] + q0, d);
#pragma unroll
          for (int v = 0; v < V; ++v) {
            const T b = cp(0, 0, si0 + v), c = cp(0, 1, si0 + v) * p.idx_, km = (cp(0, 2, si0 + v) - T(1)) * p.idx_;
            a[v] = b * a[v] + c * dHz_x[v]; d[v] = b * d[v] + c * dHy_x[v];
            ay[v] -= km * dHz_x[v] + a[v]; az[v] += km * dHy_x[v] + d[v];
          }
          stv(p.psi[pEyx] + q0, a); stv(p.psi[pEzx] + q0, d);
        }
      }
      if (owned) {
        T ex[V], ey[V];
        if (kFull) {
          T ca[V], cb[V];
          ldv(p.Ca[0] + o, ca); ldv(p.Cb[0] + o, cb);
#pragma unroll
          for (int v = 0; v < V; ++v) ex[v] = fma(cb[v], ax[v], ca[v] * ex0[v]);
          ldv(p.Ca[1] + o, ca); ldv(p.Cb[1] + o, cb);
#pragma unroll
          for (int v = 0; v < V; ++v) ey[v] = fma(cb[v], ay[v], ca[v] * ey0[v]);
          ldv(p.Ca[2] + o, ca); ldv(p.Cb[2] + o, cb);
#pragma unroll
          for (int v = 0; v < V; ++v) ez[v] = fma(cb[v], az[v], ca[v] * ez[v]);
        } else {
#pragma unroll
          for (int v = 0; v < V; ++v) {
            const Vec4<T> a = lds4(tab + 8 * (int)mi[v]), b = lds4(tab + 8 * (int)mi[v] + 4);
            ex[v] = fma(a.d, ax[v], a.a * ex0[v]);
            ey[v] = fma(b.a, ay[v], a.b * ey0[v]);
            ez[v] = fma(b.b, az[v], a.c * ez[v]);
          }
        }
        // PEC walls: low-face tangential E stays zero (R1)
        if (k == 0) {
#pragma unroll
          for (int v = 0; v < V; ++v) { ex[v] = T(0); ey[v] = T(0); }
        }
        if (wj) {
#pragma unroll
          for (int v = 0; v < V; ++v) { ex[v] = T(0); ez[v] = T(0); }
        }
        if (wi) { ey[0] = T(0); ez[0] = T(0); }
        if (xtail) {  // pad columns i >= nx stay zero: they are the high-face PEC wall (R1)
#pragma unroll
          for (int v = 0; v < V; ++v) if (v >= nvalid) { ex[v] = T(0); ey[v] = T(0); ez[v] = T(0); }
        }
        stv_stream(p.dst[kEx] + o, ex); stv_stream(p.dst[kEy] + o, ey); stv_stream(p.dst[kEz] + o, ez);
      }
    } else {
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[s]);
    }
#pragma unroll
    for (int v = 0; v < V; ++v) { ex0[v] = ex1[v]; ey0[v] = ey1[v]; exj0[v] = exj1[v]; }
    eyi0 = eyi1;
    if (it >= 1) {
#pragma unroll
      for (int v = 0; v < V; ++v) { hxm[v] = hx[v]; hym[v] = hy[v]; }
    }
    if (++s == NS) { s = 0; ph ^= 1u; }
  }
}

}  // namespace fdtd_b200
