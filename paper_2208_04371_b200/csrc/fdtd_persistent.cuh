// fdtd_persistent.cuh -- many leapfrog steps in ONE cooperative launch, for grids that live in L2.
//
// Grids such as C0 (1.5 MB) and C1 (14 MB) are not HBM-bound: a step of four tiny kernels costs four launch latencies
// (about 4 us each inside a CUDA graph: 16 us for C0's 32^3 cells).  Here one resident grid of blocks walks the whole
// grid with a grid-stride loop and separates the half steps with grid-wide barriers instead of kernel boundaries:
//
//   step n:  [H phase: H^{n+1/2} from E^n            | probe blocks: V of step n-1 (E is read-only here)]
//            grid barrier
//            [E phase: E^{n+1} from H^{n+1/2}, source | probe blocks: I of step n   (H is read-only here)]
//            grid barrier
//   after the last step: V probe of that step.
// The probes of port p are taken by a block of their own (the last `probe_blocks` blocks of the grid do nothing else) where
// the resident grid has room for it: a block that sums a port, evaluates its 2 x nf sines in fp64 AND updates its share of
// the cells would be the last one at every barrier.  Without room (probe_blocks = 0) blocks 0..ports-1 do both.
//
// The arithmetic is the two-pass step's (update_H_vec / update_E_vec of fdtd_kernels.cuh), the source is added by the
// thread that owns the cell right after its E update (ports in order, like the per-port k_source launches), and the probe
// sums use the thread -> warp -> block order of k_probe_dft's one-block path.
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>

#include "fdtd_kernels.cuh"
#include "fdtd_params.h"

namespace fdtd_b200 {

constexpr int kPersistThreads = 256;
constexpr int kPersistMaxSrc = 8;

// block-wide sum in k_probe_dft's order (per-thread strided partial, xor-shuffle per warp, warps in order)
__device__ __forceinline__ double block_sum_256(double v, double* sh) {
  v = warp_sum(v);
  __syncthreads();   // sh may still be read from the previous call
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
  __syncthreads();
  double a = 0.0;
#pragma unroll
  for (int q = 0; q < kPersistThreads / 32; ++q) a += sh[q];
  return a;
}

// V of one port from E^{n} (Eq. 4 line 1) and its DFT terms at time n dt (R7, R8); whole block
template <typename T>
__device__ __forceinline__ void probe_V_dft(const PortParams<T>& p, int port, long long n, double* sh) {
  const PortDev q = p.ports[port];
  const int nj = q.vj1 - q.vj0 + 1, nv = nj * (q.vk1 - q.vk0);
  double sv = 0.0;
  for (int s = threadIdx.x; s < nv; s += kPersistThreads) {
    const int j = q.vj0 + s % nj, k = q.vk0 + s / nj;
    sv += (double)p.Ez[q.ip + (long long)p.P * j + p.PS * k];
  }
  const double V = p.dz / (double)nj * block_sum_256(sv, sh);
  if (threadIdx.x == 0) p.lastV[port] = V;
  const double t = (double)n * p.dt;
  for (int m = threadIdx.x; m < p.nf; m += kPersistThreads) {
    double s, c;
    sincos(2.0 * 3.14159265358979323846 * p.freqs[m] * t, &s, &c);
    double* acc = p.dftV + ((long long)port * p.nf + m) * 2;
    acc[0] += V * p.dt * c;
    acc[1] -= V * p.dt * s;
  }
}

// I of one port from H^{n-1/2} (Eq. 4 line 2) and its DFT terms at time (n - 1/2) dt; whole block
template <typename T>
__device__ __forceinline__ void probe_I_dft(const PortParams<T>& p, int port, long long n, double* sh) {
  const PortDev q = p.ports[port];
  const int nkl = q.lk1 - q.lk0 + 1, njl = q.lj1 - q.lj0 + 1;
  double si = 0.0;
  for (int s = threadIdx.x; s < nkl + njl; s += kPersistThreads) {
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
  const double I = block_sum_256(si, sh);
  if (threadIdx.x == 0) p.lastI[port] = I;
  const double t = ((double)n - 0.5) * p.dt;
  for (int m = threadIdx.x; m < p.nf; m += kPersistThreads) {
    double s, c;
    sincos(2.0 * 3.14159265358979323846 * p.freqs[m] * t, &s, &c);
    double* acc = p.dftI + ((long long)port * p.nf + m) * 2;
    acc[0] += I * p.dt * c;
    acc[1] -= I * p.dt * s;
  }
}

struct SrcBox { int is, sj0, sj1, sk0, sk1, port; };

template <typename T, int MODE>
__global__ void __launch_bounds__(kPersistThreads) k_steps_persistent(const StepParams<T> p, const PortParams<T> q, int nsteps,
                                                                      int probe_blocks) {
  namespace cg = cooperative_groups;
  cg::grid_group grid = cg::this_grid();
  constexpr int V = VecOf<T>::V;
  __shared__ double sh[kPersistThreads / 32];
  __shared__ SrcBox sbox[kPersistMaxSrc];
  __shared__ T sg[kPersistMaxSrc];
  __shared__ int nsrc_s;

  if (threadIdx.x == 0) {
    int n = 0;
    for (int t = 0; t < q.nports && n < kPersistMaxSrc; ++t) {
      const PortDev d = q.ports[t];
      if (d.has_source) { sbox[n] = SrcBox{d.is, d.sj0, d.sj1, d.sk0, d.sk1, t}; ++n; }
    }
    nsrc_s = n;
  }
  __syncthreads();
  const int nsrc = nsrc_s;
  const int nvx = (p.nx + V - 1) / V;
  const int nvec = nvx * p.ny * p.nz;                       // the host uses this kernel below 2^31 vectors only
  const int nfb = (int)gridDim.x - probe_blocks;            // blocks that update cells
  const bool field_block = (int)blockIdx.x < nfb;
  // ports this block probes: block b of the probe blocks takes ports b, b + probe_blocks, ...; shared duty: b, b + gridDim.x, ...
  const int port0 = probe_blocks > 0 ? (int)blockIdx.x - nfb : (int)blockIdx.x, port_step = probe_blocks > 0 ? probe_blocks : (int)gridDim.x;
  const int tid0 = field_block ? blockIdx.x * kPersistThreads + threadIdx.x : 0x7fffffff, nthr = nfb * kPersistThreads;
  const long long n0 = *p.nstep;                            // written again only after the last grid barrier

  for (int s = 0; s < nsteps; ++s) {
    const long long n = n0 + s + 1;                         // this step ends at t = n dt
    // ---- H phase ----------------------------------------------------------------------------------------------------
    if (threadIdx.x < nsrc) {                               // source amplitudes of this step, read after the barrier below
      const PortDev d = q.ports[sbox[threadIdx.x].port];
      sg[threadIdx.x] = (T)(d.amp * waveform_dev(d.waveform, (double)n * q.dt, d.t0, d.sigma, d.f0));
    }
    if (s > 0 && port0 >= 0)
      for (int port = port0; port < q.nports; port += port_step) probe_V_dft(q, port, n - 1, sh);
    for (int v = tid0; v < nvec; v += nthr) {
      const int iv = v % nvx, jk = v / nvx;
      update_H_vec<T, MODE>(p, iv * V, jk % p.ny, jk / p.ny);
    }
    grid.sync();
    // ---- E phase, source ----------------------------------------------------------------------------------------------
    if (port0 >= 0)
      for (int port = port0; port < q.nports; port += port_step) probe_I_dft(q, port, n, sh);
    for (int v = tid0; v < nvec; v += nthr) {
      const int iv = v % nvx, jk = v / nvx;
      const int i0 = iv * V, j = jk % p.ny, k = jk / p.ny;
      update_E_vec<T, MODE>(p, i0, j, k);
      for (int t = 0; t < nsrc; ++t) {
        const SrcBox b = sbox[t];
        if (k >= b.sk0 && k < b.sk1 && j >= b.sj0 && j <= b.sj1 && b.is >= i0 && b.is < i0 + V)
          q.Ez[b.is + (long long)p.P * j + p.PS * k] += sg[t];
      }
    }
    grid.sync();
  }
  if (port0 >= 0)
    for (int port = port0; port < q.nports; port += port_step) probe_V_dft(q, port, n0 + nsteps, sh);
  if (blockIdx.x == 0 && threadIdx.x == 0) *p.nstep = n0 + nsteps;
}

}  // namespace fdtd_b200
