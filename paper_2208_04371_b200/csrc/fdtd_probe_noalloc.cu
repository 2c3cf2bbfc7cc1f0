// fdtd_probe_noalloc.cu -- fdtd_port_probe_noalloc(): the port voltage / current integrals of Eq. 4 (reading
// R7) for a caller that has nowhere to take device memory from.
//
// Why this exists.  Everything else in this library works out of a workspace the caller allocates and hands to
// fdtd_commit().  Some users of the probes cannot do that: a monitor thread that looks at the fields of a run in flight
// (an allocation call synchronises the whole device and would stall the time stepping it is watching), a plug-in inside a host
// program that gave all of the GPU's memory to its own pool at start-up (an allocation there simply fails), a diagnostic
// hook that runs while the surrounding program forbids allocator calls.  They do own the field arrays they want probed and
// a few bytes for the answer; what they lack is the few KB of hand-over memory the multi-block reduction needs between its
// blocks.  Here that memory is part of the library image: a fixed array in device memory that every GPU receives when it
// loads the library and keeps until the process ends (kScratchBytes below, about 16 KB per GPU).
//
// The kernel is the reduction of k_probe_dft (fdtd_kernels.cuh) without its DFT tail, on the caller's plain nx*ny*nz arrays,
// and ALWAYS with the hand-over through the scratch array (the handle-based kernel skips it for one-block ports).  This file
// shares no state with the handle-based path and changes nothing in it.
//
// Rules that follow from the shared array (also in include/fdtd.h):
//   * sizes are capped: FDTD_NOALLOC_MAX_PORTS ports per call; more is refused with FDTD_ERANGE, nothing is enqueued;
//   * the array keeps what the previous call left.  The per-port arrival counters must be zero when the kernel starts, so each
//     call clears them on the stream first (a kernel that was cut short would otherwise poison every later call); the partial
//     sums need no clearing, every slot that is read has been written by the same launch;
//   * two calls whose kernels can run at the same time on one GPU (different streams, different host threads) use the same
//     counters and slots and corrupt each other.  Calls on one stream are ordered and safe;
//   * the first call on a GPU asks the runtime where that GPU's copy of the array lives (cudaGetSymbolAddress) and remembers
//     the answer; make that first call outside any stream capture.
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "../../include/fdtd.h"

namespace {

constexpr int kThreads = 256;
constexpr int kMaxPorts = FDTD_NOALLOC_MAX_PORTS;
constexpr int kMaxBlocks = FDTD_NOALLOC_MAX_BLOCKS;
constexpr int kMaxDevices = 64;
// scratch layout: partial sums [port][block][V, I] as doubles, then one arrival counter per port
constexpr size_t kPartialBytes = sizeof(double) * 2 * kMaxBlocks * kMaxPorts;
constexpr size_t kCounterBytes = 256;   // kMaxPorts ints, rounded up so that the array stays a whole number of 256-byte lines
constexpr size_t kScratchBytes = kPartialBytes + kCounterBytes;
static_assert(sizeof(int) * kMaxPorts <= kCounterBytes, "counters do not fit their slot");
static_assert(kScratchBytes == FDTD_NOALLOC_SCRATCH_BYTES, "include/fdtd.h states another scratch size");

// The scratch itself.  One copy per GPU that loads this library, alive until the process exits.  In HOST code this name is only
// a handle for the runtime (its host-side value is not a device address): the host passes the kernels the address that
// cudaGetSymbolAddress returned for the current device, never `g_scratch` itself.
static __device__ __align__(256) unsigned char g_scratch[kScratchBytes];

struct ProbePort { int ip, vj0, vj1, vk0, vk1, lj0, lj1, lk0, lk1; };
struct ProbeArgs {
  ProbePort port[kMaxPorts];
  int nx;
  long long plane;   // nx * ny
  double dy, dz;
};

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int s = 16; s > 0; s >>= 1) v += __shfl_xor_sync(0xffffffffu, v, s);
  return v;
}

// grid (nblk, nports).  Every block writes the partial V and I sums of its slice into its slot of the scratch; the block that
// arrives last at the port's counter adds the slots in block order (so the answer does not depend on which block that was),
// writes V and I of the port and puts the counter back to zero.
//   V = (dz / n_col) * sum Ez over the V box;   I = dz * sum_k (Hz[lj1,k] - Hz[lj0-1,k]) - dy * sum_j (Hy[j,lk1] - Hy[j,lk0-1])
template <typename T>
__global__ void __launch_bounds__(kThreads) k_probe_noalloc(const T* __restrict__ Ez, const T* __restrict__ Hy,
                                                            const T* __restrict__ Hz, const ProbeArgs a, double* partial,
                                                            int* counter, double* __restrict__ VI) {
  __shared__ double sh[2][kThreads / 32];
  const int port = blockIdx.y, nblk = gridDim.x;
  const ProbePort q = a.port[port];
  const long long P = a.nx, PS = a.plane;
  const int gtid = blockIdx.x * kThreads + threadIdx.x, gstride = nblk * kThreads;
  const int nj = q.vj1 - q.vj0 + 1, nv = nj * (q.vk1 - q.vk0);
  double sv = 0.0;
  for (int s = gtid; s < nv; s += gstride) {
    const int j = q.vj0 + s % nj, k = q.vk0 + s / nj;
    sv += (double)Ez[q.ip + P * j + PS * k];
  }
  const int nkl = q.lk1 - q.lk0 + 1, njl = q.lj1 - q.lj0 + 1;
  double si = 0.0;
  for (int s = gtid; s < nkl + njl; s += gstride) {
    if (s < nkl) {
      const int k = q.lk0 + s;
      si += a.dz * ((double)Hz[q.ip + P * q.lj1 + PS * k] - (double)Hz[q.ip + P * (q.lj0 - 1) + PS * k]);
    } else {
      const int j = q.lj0 + (s - nkl);
      si -= a.dy * ((double)Hy[q.ip + P * j + PS * q.lk1] - (double)Hy[q.ip + P * j + PS * (q.lk0 - 1)]);
    }
  }
  sv = warp_sum(sv); si = warp_sum(si);
  if ((threadIdx.x & 31) == 0) { sh[0][threadIdx.x >> 5] = sv; sh[1][threadIdx.x >> 5] = si; }
  __syncthreads();
  if (threadIdx.x != 0) return;
  double v = 0.0, i = 0.0;
#pragma unroll
  for (int w = 0; w < kThreads / 32; ++w) { v += sh[0][w]; i += sh[1][w]; }
  double* slot = partial + ((long long)port * kMaxBlocks + blockIdx.x) * 2;
  slot[0] = v; slot[1] = i;
  __threadfence();
  if (atomicAdd(counter + port, 1) != nblk - 1) return;
  __threadfence();
  const volatile double* all = partial + (long long)port * kMaxBlocks * 2;
  double V = 0.0, I = 0.0;
  for (int b = 0; b < nblk; ++b) { V += all[2 * b]; I += all[2 * b + 1]; }
  VI[2 * port] = V * (a.dz / (double)nj);
  VI[2 * port + 1] = I;
  counter[port] = 0;
}

// Address of g_scratch on each device, filled in by the first call that runs on it.
std::mutex g_setup_lock;
unsigned char* g_scratch_on[kMaxDevices] = {};

int fail(char* errbuf, size_t len, int code, const char* fmt, ...) {
  if (errbuf && len) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(errbuf, len, fmt, ap);
    va_end(ap);
  }
  return code;
}

// device a pointer lives on; -1 unless it is plain device memory
int device_memory_of(const void* p) {
  cudaPointerAttributes at;
  if (!p || cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return -1; }
  return at.type == cudaMemoryTypeDevice ? at.device : -1;
}

struct OnDevice {   // make `dev` current for the duration of the call, then give the caller's device back
  int prev = -1;
  bool switched = false;
  bool ok = false;
  explicit OnDevice(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) { cudaGetLastError(); return; }
    if (prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
    ok = prev == dev || switched;
  }
  ~OnDevice() { if (switched) cudaSetDevice(prev); }
};

}  // namespace

extern "C" int fdtd_port_probe_noalloc(const void* Ez, const void* Hy, const void* Hz, int precision, int nx, int ny, int nz,
                                       double dy, double dz, const fdtd_port* ports, int nports, double* VI,
                                       void* cuda_stream, char* errbuf, size_t errbuf_len) {
  if (errbuf && errbuf_len) errbuf[0] = 0;
  if (precision != FDTD_F32 && precision != FDTD_F64)
    return fail(errbuf, errbuf_len, FDTD_EINVAL, "fdtd_port_probe_noalloc: precision must be FDTD_F32 or FDTD_F64");
  if (nx < 2 || ny < 2 || nz < 2 || !(dy > 0) || !(dz > 0) || !ports || nports < 1)
    return fail(errbuf, errbuf_len, FDTD_EINVAL, "fdtd_port_probe_noalloc: bad grid, cell size or port list");
  if (nports > kMaxPorts)
    return fail(errbuf, errbuf_len, FDTD_ERANGE,
                "fdtd_port_probe_noalloc: %d ports asked for, the built-in scratch serves at most %d per call (split the list)",
                nports, kMaxPorts);
  if ((long long)ny * nz > 0x7fffffffLL)   // the kernel numbers the samples of a port box with an int
    return fail(errbuf, errbuf_len, FDTD_ERANGE, "fdtd_port_probe_noalloc: ny * nz does not fit 31 bits");
  ProbeArgs a{};
  a.nx = nx; a.plane = (long long)nx * ny; a.dy = dy; a.dz = dz;
  auto in = [](int v, int lo, int hi) { return v >= lo && v < hi; };
  long long most = 1;
  for (int n = 0; n < nports; ++n) {
    const fdtd_port& p = ports[n];
    if (!(in(p.ip, 0, nx) && in(p.vj0, 0, ny) && in(p.vj1, p.vj0, ny) && in(p.vk0, 0, nz) && p.vk1 > p.vk0 && p.vk1 <= nz))
      return fail(errbuf, errbuf_len, FDTD_ERANGE, "fdtd_port_probe_noalloc: port %d: voltage box outside the grid", n);
    if (!(in(p.lj0, 1, ny) && in(p.lj1, p.lj0, ny) && in(p.lk0, 1, nz) && in(p.lk1, p.lk0, nz)))
      return fail(errbuf, errbuf_len, FDTD_ERANGE,
                  "fdtd_port_probe_noalloc: port %d: current loop outside the grid (needs lj0 >= 1, lk0 >= 1)", n);
    a.port[n] = ProbePort{p.ip, p.vj0, p.vj1, p.vk0, p.vk1, p.lj0, p.lj1, p.lk0, p.lk1};
    const long long nv = (long long)(p.vj1 - p.vj0 + 1) * (p.vk1 - p.vk0);
    const long long nl = (long long)(p.lj1 - p.lj0 + 1) + (p.lk1 - p.lk0 + 1);
    most = nv > most ? nv : most;
    most = nl > most ? nl : most;
  }
  const int dev = device_memory_of(Ez);
  if (dev < 0 || device_memory_of(Hy) != dev || device_memory_of(Hz) != dev || device_memory_of(VI) != dev)
    return fail(errbuf, errbuf_len, FDTD_EINVAL, "fdtd_port_probe_noalloc: Ez, Hy, Hz and VI must be device memory of one GPU");
  if (dev >= kMaxDevices)
    return fail(errbuf, errbuf_len, FDTD_ERANGE, "fdtd_port_probe_noalloc: device ordinal %d beyond %d", dev, kMaxDevices - 1);
  OnDevice cur(dev);
  if (!cur.ok) return fail(errbuf, errbuf_len, FDTD_ECUDA, "fdtd_port_probe_noalloc: cannot make device %d current", dev);
  cudaError_t e;
  unsigned char* scratch;
  {
    // set-up, once per GPU, with that GPU current: where does its copy of g_scratch live?
    std::lock_guard<std::mutex> hold(g_setup_lock);
    if (!g_scratch_on[dev]) {
      unsigned char* ptr = nullptr;
      if ((e = cudaGetSymbolAddress((void**)&ptr, g_scratch)) != cudaSuccess || !ptr) {
        cudaGetLastError();
        return fail(errbuf, errbuf_len, FDTD_ECUDA, "fdtd_port_probe_noalloc: cudaGetSymbolAddress on device %d: %s", dev,
                    cudaGetErrorString(e));
      }
      g_scratch_on[dev] = ptr;
    }
    scratch = g_scratch_on[dev];
  }
  double* partial = reinterpret_cast<double*>(scratch);
  int* counter = reinterpret_cast<int*>(scratch + kPartialBytes);
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  // the counters must read zero when the kernel starts, whatever an earlier call left behind
  if ((e = cudaMemsetAsync(counter, 0, kCounterBytes, stream)) != cudaSuccess) {
    cudaGetLastError();
    return fail(errbuf, errbuf_len, FDTD_ECUDA, "fdtd_port_probe_noalloc: clearing the counters: %s", cudaGetErrorString(e));
  }
  long long nblk = (most + kThreads - 1) / kThreads;
  if (nblk > kMaxBlocks) nblk = kMaxBlocks;   // the slices are strided: 64 blocks take any box
  const dim3 grid((unsigned)nblk, (unsigned)nports, 1);
  if (precision == FDTD_F64)
    k_probe_noalloc<double><<<grid, kThreads, 0, stream>>>(static_cast<const double*>(Ez), static_cast<const double*>(Hy),
                                                           static_cast<const double*>(Hz), a, partial, counter, VI);
  else
    k_probe_noalloc<float><<<grid, kThreads, 0, stream>>>(static_cast<const float*>(Ez), static_cast<const float*>(Hy),
                                                          static_cast<const float*>(Hz), a, partial, counter, VI);
  if ((e = cudaGetLastError()) != cudaSuccess)
    return fail(errbuf, errbuf_len, FDTD_ECUDA, "fdtd_port_probe_noalloc: launch: %s", cudaGetErrorString(e));
  return FDTD_OK;
}
