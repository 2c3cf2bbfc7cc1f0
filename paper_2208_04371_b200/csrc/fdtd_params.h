// fdtd_params.h -- plain-data descriptors handed by value from the host plan (fdtd_api.cu) to the kernels.
//
// HBM layout: every per-cell array (six field components, the uint8 material index, the
// full-mode coefficient arrays) uses ONE padded geometry so that a single offset serves them all and every
// out-of-range stencil operand is an in-bounds zero:
//     element (i,j,k)  ->  base + i + P*(j + R*(k+1)),   P = round_up(nx+1, 128 B),  R = ny+1,  nz+2 planes.
// Row ny of every plane, the columns i >= nx of every row and the planes -1 and nz are zero and are never written:
// they are the PEC wall behind everything (high-face tangential E "not stored, reads as 0"; H outside the box reads
// as 0 for the low-face E rows, which are then forced to 0 anyway; include/fdtd.h "Walls").
// Pointers in these structs already point at element (0,0,0).
#pragma once
#include <stdint.h>

namespace fdtd_b200 {

enum { kEx = 0, kEy, kEz, kHx, kHy, kHz };
// order of the 12 psi arrays (name = component, derivative axis)
enum { pHxy = 0, pHzy, pHxz, pHyz, pHyx, pHzx, pExy, pEzy, pExz, pEyz, pEyx, pEzx };

constexpr int kMaxTable = 256;
constexpr int kMaxSlab = 64;   // fused kernel: CPML cells per axis (lo + hi) whose coefficient vectors fit its shared memory
// material table (indexed mode), one 32-byte (fp32) / 64-byte (fp64) record per entry so that a look-up is two
// (four) 128-bit loads:  tab[8*m + 0..5] = Cax Cay Caz Cbx Cby Cbz, then tab[kTabH + 4*m + 0..2] = Dbx Dby Dbz.
constexpr int kTabH = 8 * kMaxTable;
constexpr int kTabWords = 12 * kMaxTable;

template <typename T>
struct StepParams {
  int nx, ny, nz;
  int P;            // x pitch (elements)
  long long PS;     // plane stride (elements) = P * (ny + 1)
  T* src[6];        // fields read  (Ex Ey Ez Hx Hy Hz)
  T* dst[6];        // fields written (== src for the two-pass in-place kernels)
  // materials
  const uint8_t* idx;   // indexed mode: one byte per cell, field geometry
  const T* tab;         // indexed mode: kTabWords words, layout above (kTabH)
  const T* Ca[3];       // full mode, field geometry
  const T* Cb[3];
  const T* Db[3];       // full mode with mu
  T db0;                // uniform dt/mu0 when there is no mu
  T idx_, idy_, idz_;   // 1/dx, 1/dy, 1/dz
  // CPML: thickness per face and per-axis coefficient vectors indexed by the slab coordinate s in [0, lo+hi)
  int lo[3], hi[3];
  // x slabs in whole 16-byte vectors: cells [0, xlo_end) and [xhi_begin, pitch) carry psi; padded slab coordinate
  // sp(i) = i below xlo_end, xlo_end + (i - xhi_begin) from xhi_begin on; Sxp = padded cells per row (multiple of the
  // vector length).  Cells of those vectors outside the true layer have b = 1, c = 0, 1/kappa = 1: their psi stays zero.
  int xlo_end, xhi_begin, Sxp;
  const T* bE[3]; const T* cE[3]; const T* kE[3];   // kE = 1/kappa at integer positions (E profile)
  const T* bH[3]; const T* cH[3]; const T* kH[3];   // at half-integer positions (H profile)
  T* psi[12];       // slab-only arrays: y-slab  i + P*(s + Sy*k);  z-slab  i + P*(j + ny*s);  x-slab  sp + Sxp*(j + ny*k)
  long long* nstep; // device step counter, incremented by the first kernel of every step
  int z_lo_open;    // 1: this grid is a z slab of a larger one and plane 0 is not a wall (Ex, Ey there are ordinary cells)
  // region launches of the two-pass kernels (the shell around a two-step box, fdtd_step2.cuh): ONE launch covers up to
  // kMaxRegions disjoint boxes of cells [i0, i0 + nvx * V) x [j0, j0 + ny) x [k0, k0 + nk); its 1-D grid numbers, region after
  // region, the planes of a box and within a plane the blocks over its row vectors (rows back to back: bpp blocks per plane);
  // blk0 = first block of the region.  bump = this launch increments the step counter.
  struct Region { int i0, j0, k0, nvx, ny, bpp; unsigned blk0; };
  static constexpr int kMaxRegions = 10;
  int nreg, bump;
  Region reg[kMaxRegions];
  T* peer_E[2];     // z slab linked to its lower neighbour (fdtd_z_link): that slab's halo plane nz of Ex, Ey (element (0,0)
                    // of the plane, same pitch), written by the kernel that updates E on plane 0; nullptr = not linked
};

struct PortDev {
  int has_source;
  int is, sj0, sj1, sk0, sk1;
  int waveform;
  double amp, t0, sigma, f0;
  int ip;
  int vj0, vj1, vk0, vk1;
  int lj0, lj1, lk0, lk1;
};

template <typename T>
struct PortParams {
  int P;
  long long PS;
  T* Ez; const T* Hy; const T* Hz;
  const PortDev* ports;
  int nports;
  const double* freqs;
  int nf;
  double* dftV;   // [port][freq][re,im]
  double* dftI;
  double* lastV;  // [port]
  double* lastI;
  double* partial;  // [port][kProbeMaxBlocks][V, I] per-block partial sums of k_probe_dft
  int* pcount;      // [port] blocks of k_probe_dft that have delivered their partial; returns to 0 every step
  const long long* nstep;  // already incremented: E time = nstep*dt, H time = (nstep - 1/2)*dt
  double dt, dy, dz;
};

}  // namespace fdtd_b200
