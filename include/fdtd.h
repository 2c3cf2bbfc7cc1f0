/* fdtd.h -- C ABI of the B200-native explicit Yee FDTD hot path (arXiv 2208.04371, ARTEMIS S-parameter workflow).
 *
 * What the library computes (citations: PAPER.md = /root/reference/PAPER.md; R* = readings in DESIGN.md):
 *   one leapfrog time step  H^{n-1/2} -> H^{n+1/2},  E^n -> E^{n+1}  of the "conventional FDTD" on a Yee grid
 *    with per-cell permittivity / conductivity / permeability coefficients,
 *   PEC walls and PEC/lossy metal, an absorbing layer on chosen faces (realised as
 *   CPML, R4), the soft port source of Eq. 3, the port voltage and current integrals of Eq. 4
 *    and the DFT of their histories accumulated on the device every step.
 *   S* (Eq. 1-2) is formed by the caller from fdtd_read_port_dft() of an "inc" and a "tot" run.
 *
 * Conventions
 *   Grid      nx*ny*nz Yee cells, x fastest.  Cell (i,j,k) owns the samples
 *               Ex(i+1/2,j,k) Ey(i,j+1/2,k) Ez(i,j,k+1/2) Hx(i,j+1/2,k+1/2) Hy(i+1/2,j,k+1/2) Hz(i+1/2,j+1/2,k)   (R1)
 *             Caller-visible arrays hold exactly N = nx*ny*nz elements, index i + nx*(j + ny*k).  Propagation axis of
 *             the ports is x, "vertical" is z (the paper uses y and z; a relabelling).
 *   Walls     all six outer faces are PEC, behind any CPML.  Low-face tangential E is stored and forced to 0;
 *             high-face tangential E is not stored and reads as 0 (R1).
 *   Time      after n steps the E arrays hold E at t = n*dt, the H arrays hold H at t = (n-1/2)*dt (R5).
 *   Pointers  every pointer argument documented "host or device" may be either; the library asks the CUDA runtime
 *             which.  All other pointers are host pointers.  Nothing is retained after a call returns except the
 *             workspace given to fdtd_commit().
 *   Memory    the CALLER owns all device memory: one buffer of fdtd_workspace_bytes() bytes (256-byte aligned), and
 *             a CUDA stream.  The library never allocates device memory.  (The one piece of device memory that is the
 *             library's own is the fixed FDTD_NOALLOC_SCRATCH_BYTES array inside its image that fdtd_port_probe_noalloc uses;
 *             see the end of this file.)
 *   Errors    every int-returning call returns FDTD_OK (0) or a negative code; fdtd_last_error() gives a message.
 *             No exceptions, no abort, no printing.  There is NO CPU fallback: without a CUDA device
 *             fdtd_commit() fails with FDTD_ECUDA.
 *   Lifecycle fdtd_create -> {fdtd_set_boundary, fdtd_set_material_mode, fdtd_add_port, fdtd_set_dft,
 *             fdtd_set_option} in any order -> fdtd_workspace_bytes -> fdtd_commit -> {fdtd_set_materials_*,
 *             fdtd_step, fdtd_read_*, fdtd_write_fields, fdtd_reset} -> fdtd_destroy.
 *             Calling out of order returns FDTD_ESTATE.  A freshly committed object is vacuum, all state zero.
 *   Device    a handle belongs to the device its workspace lives on (fdtd_commit asks the runtime).  Every later call
 *             makes that device current for its own duration and restores the caller's, so a handle committed on
 *             device 1 may be driven while device 0 is current.  The stream given to fdtd_commit must be one of that
 *             device.
 *   Threads   one handle must not be used from two host threads at once.
 */
#ifndef FDTD_B200_H
#define FDTD_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fdtd fdtd_t; /* opaque host object owned by the library */

enum { FDTD_OK = 0, FDTD_EINVAL = -1, FDTD_ECFL = -2, FDTD_ESTATE = -3, FDTD_ENOMEM = -4, FDTD_ECUDA = -5, FDTD_ERANGE = -6 };
enum { FDTD_F32 = 32, FDTD_F64 = 64 };
enum { FDTD_W_DGAUSS = 0 /* Eq. 3 */, FDTD_W_GAUSS = 1, FDTD_W_GSINE = 2 };
enum { FDTD_MAT_INDEXED = 0, FDTD_MAT_FULL = 1 };
enum { FDTD_EX = 0, FDTD_EY, FDTD_EZ, FDTD_HX, FDTD_HY, FDTD_HZ };

/* Options for fdtd_set_option (before commit). */
enum {
  FDTD_OPT_STEP_IMPL = 1,   /* 0 = auto: fdtd_commit measures the candidates on the committed all-zero state and keeps the
                                   fastest (below 4 Mi cells: two-pass vs persistent; above: two-pass vs fused; from 8 Mi
                                   cells also 4, where the grid leaves it a box),
                               1 = two-pass (H kernel, E kernel, in place),
                               2 = fused E+H kernel (temporal blocking over the half steps; a second field set),
                               3 = persistent: fdtd_step(n) is one cooperative launch per 4096 steps, with grid-wide
                                   barriers between the half steps (grids that live in L2; the arithmetic of 1),
                               4 = two steps per pass: a box of cells that keeps two cells' distance from the CPML
                                   layers is advanced TWO steps by one kernel (every field read and written once per two
                                   steps; the kernel adds the first step's source itself), the shell around it -- and a
                                   band of cells around every port plane inside the box, for the probes of the first
                                   step -- step by step with the kernels of 1; at most 4 driving ports; fdtd_commit
                                   returns FDTD_EINVAL when the grid leaves no such box; a second field set */
  FDTD_OPT_USE_GRAPH = 2,   /* 1 (default) = replay a captured CUDA graph per FDTD_OPT_GRAPH_UNROLL steps; 0 = plain launches.
                               Capture needs a real stream: on the NULL (legacy default) stream fdtd_step always issues
                               plain launches (fdtd_graph_replays() stays 0)                                             */
  FDTD_OPT_GRAPH_UNROLL = 3,/* steps per captured graph (default 8; rounded up to even for the fused step)              */
  FDTD_OPT_FUSED_KZ = 4,    /* planes per z chunk of the fused kernel (0 = auto: measured at commit)                    */
  FDTD_OPT_Z_SPIN = 5,      /* linked z slabs: polls of a hand-over counter before a wait gives up (default 2e7; a poll sleeps
                               about 1 us, so about 20 s).  After the first time-out the slab's later waits return at once    */
  FDTD_OPT_FUSED_TILE = 6,  /* tile of the fused kernel: 0 = auto (measured at commit), 1 = 128 x 14 cells (fp64: 64 x 14), one
                               block per SM; 2 = 128 x 6 (64 x 6), two blocks per SM: twice the tiles and two z marches per
                               SM for mid-size grids.  The results are the same cell by cell whatever the tile            */
  FDTD_OPT_TUNE_MEMO = 7    /* 1 (default) = what fdtd_commit measured for a configuration (device, precision, grid, material
                               mode, CPML thicknesses, STEP_IMPL / FUSED_KZ / FUSED_TILE, z interfaces, port / source /
                               frequency counts) is remembered for the life of the process and taken again, unmeasured, by
                               every later commit of the same configuration: one program always runs one implementation.
                               0 = measure afresh.  Reproducibility: results are bit-identical for a given implementation,
                               tile and chunk length (fdtd_impl_name, fdtd_fused_kz, fdtd_fused_tile report them); between
                               implementations they agree to the parity tolerance only (different fma / summation order), and
                               with two steps per pass (4, or 0 where it is selected) an odd fdtd_step(n) runs its last step
                               with the one-step kernels -- so how a caller batches its steps is part of that configuration.
                               Across processes the automatic choice may differ: pin it with FDTD_OPT_STEP_IMPL / FUSED_KZ /
                               FUSED_TILE from a reported run where bitwise repeatability matters                             */
};

/* A port (Fig. 1a): a soft E_z source on a box of the plane i = is (surface 'e'), a voltage box and
 * a current loop on the plane i = ip.
 *   source   E_z[is, j, k] += amp * g((n+1)*dt)   for j in sj0..sj1 (inclusive), k in [sk0, sk1)          (R6, R8)
 *            g: DGAUSS -2u exp(-u^2) (Eq. 3) | GAUSS exp(-u^2) | GSINE sin(2 pi f0 (t-t0)) exp(-u^2), u = (t-t0)/sigma
 *   V        (dz / (vj1-vj0+1)) * sum_{j=vj0..vj1} sum_{k=vk0..vk1-1} E_z[ip, j, k]                        (Eq. 4, R7)
 *   I        dz * sum_{k=lk0..lk1} (Hz[ip,lj1,k] - Hz[ip,lj0-1,k]) - dy * sum_{j=lj0..lj1} (Hy[ip,j,lk1] - Hy[ip,j,lk0-1])
 *            -- the discrete Ampere loop, right-handed about +x, one cell away from metal occupying node columns
 *            lj0+1..lj1-1 and planes lk0+1..lk1-1.  Needs lj0 >= 1 and lk0 >= 1.           (R7)
 */
typedef struct fdtd_port {
  int has_source;
  int is, sj0, sj1, sk0, sk1;
  int waveform;
  double amp, t0, sigma, f0;
  int ip;
  int vj0, vj1, vk0, vk1;
  int lj0, lj1, lk0, lk1;
} fdtd_port;

/* Create a solver for an nx*ny*nz grid with cell size (dx,dy,dz) [m] and time step dt [s]; precision = FDTD_F32|F64
 * is the arithmetic and storage type of the fields.  FDTD_ECFL if dt > 1/(c*sqrt(1/dx^2+1/dy^2+1/dz^2)) (PAPER.md:93,
 * 116 run at 0.9 of it); FDTD_EINVAL if any n < 2, any d <= 0, dt <= 0 or a bad precision.  *out is set on success. */
int fdtd_create(int nx, int ny, int nz, double dx, double dy, double dz, double dt, int precision, fdtd_t** out);

/* CPML thickness in cells on the faces x-,x+,y-,y+,z-,z+ (0 = bare PEC wall; PML on every face but the
 * ground).  cpml = NULL for defaults or {m, m_a, kappa_max, alpha_max, sigma_factor, eps_r_pml} (R4):
 * sigma_max = sigma_factor*(m+1)/(eta0*d_axis*sqrt(eps_r_pml)).  FDTD_ERANGE if lo+hi > n on an axis. */
int fdtd_set_boundary(fdtd_t*, const int pml_cells[6], const double* cpml);

/* Declare how materials will be given after commit (decides the workspace size).  Default: INDEXED, has_mu = 0.
 *   FDTD_MAT_INDEXED  one uint8 per cell into a table of <= 256 entries (a handful of materials)
 *   FDTD_MAT_FULL     per-cell, per-component arrays (anisotropic eps_xx/yy/zz, sigma_xx/yy/zz)
 * has_mu != 0 reserves room for per-entry / per-cell permeability. */
int fdtd_set_material_mode(fdtd_t*, int mode, int has_mu);

/* Add a port; *port_id (may be NULL) receives its index.  FDTD_ERANGE if a sample lies outside the grid, or if the source
 * box touches the plane i = 0 or the row j = 0: E_z there is a PEC wall sample that stays zero (R1). */
int fdtd_add_port(fdtd_t*, const fdtd_port* p, int* port_id);

/* Frequencies [Hz] of the running DFT of every port's V and I.  nf = 0 switches it off. */
int fdtd_set_dft(fdtd_t*, const double* freqs_hz, int nf);

int fdtd_set_option(fdtd_t*, int option, long value);

/* Bytes of device memory fdtd_commit() needs with the settings made so far. */
size_t fdtd_workspace_bytes(const fdtd_t*);

/* Adopt the caller's device buffer (device pointer, >= fdtd_workspace_bytes(), 256-byte aligned) and CUDA stream
 * (a cudaStream_t passed as void*; NULL = the legacy default stream, on which no CUDA graph can be captured), build the
 * CPML / port tables, zero all state, set vacuum everywhere.  All later work is enqueued on that stream.
 * FDTD_EINVAL also when FDTD_OPT_STEP_IMPL = 2 was asked for with more than 64 CPML cells (lo + hi) on an axis. */
int fdtd_commit(fdtd_t*, void* device_workspace, size_t bytes, void* cuda_stream);

/* Materials, component-sampled at the location of each E (eps_r, sigma) and H (mu_r) sample; the library never
 * averages (R12).  sigma = +INFINITY marks a perfect conductor.  Coefficients (R3):
 *   a = sigma*dt/(2*eps0*eps_r);  Ca = (1-a)/(1+a);  Cb = (dt/(eps0*eps_r))/(1+a);  Db = dt/(mu0*mu_r).
 * indexed: idx = N uint8, host or device; eps_r, sigma, mu_r = host arrays [n_entries][3] (x,y,z component), mu_r may
 *          be NULL (= 1) and must be NULL unless has_mu was declared.
 * full:    eps_r[c], sigma[c], mu_r[c] = arrays of N elements of the field precision, host or device; mu_r may be NULL.
 * May be called again later to change materials; fields are not touched. */
int fdtd_set_materials_indexed(fdtd_t*, const uint8_t* idx, int n_entries, const double* eps_r, const double* sigma,
                               const double* mu_r);
int fdtd_set_materials_full(fdtd_t*, const void* const eps_r[3], const void* const sigma[3], const void* const mu_r[3]);

/* Enqueue n full time steps (R5: psi_H, H; psi_E, E, walls; source; probes; DFT) on the stream.  Does not synchronise. */
int fdtd_step(fdtd_t*, long n);

/* Run n full steps exactly like fdtd_step (plain launches, no graph) with CUDA events recorded on the stream between
 * the kernels, and return the average device time per step, in milliseconds, of
 *   ms_avg[0] = H pass (or the fused E+H kernel), ms_avg[1] = E pass (0 when fused), ms_avg[2] = source injection,
 *   ms_avg[3] = probes + DFT.   This is the measurement hook of bench.py's roofline line.  Synchronises the stream.
 * With FDTD_OPT_STEP_IMPL = 4 the steps run in pairs (n is rounded up to even): ms_avg[0] = the two-step box kernel,
 * ms_avg[1] = the shell passes with their port kernels, both per step; ms_avg[2] = ms_avg[3] = 0.
 * FDTD_ESTATE on a z slab (fdtd_set_z_interfaces) or between fdtd_step_begin and fdtd_step_end. */
int fdtd_profile_step(fdtd_t*, long n, double ms_avg[4]);

/* Copy one field component (FDTD_EX..FDTD_HZ) to / from a caller array of N elements of the field precision, host or
 * device.  Stream-ordered; synchronises the stream before returning when the caller array is in host memory.
 * write_fields is the test hook for initial conditions and the resume path; FDTD_ESTATE between fdtd_step_begin and
 * fdtd_step_end (the two field sets are half updated then). */
int fdtd_read_fields(fdtd_t*, int comp, void* dst);
int fdtd_write_fields(fdtd_t*, int comp, const void* src);

/* DFT accumulators of one port: V_reim and I_reim receive 2*nf doubles (re, im interleaved), host memory.
 *   V^[m] = sum_n V^{n+1}  exp(-j 2 pi f_m (n+1)  dt) dt,   I^[m] = sum_n I^{n+1/2} exp(-j 2 pi f_m (n+1/2) dt) dt   (R8)
 * Synchronises the stream. */
int fdtd_read_port_dft(fdtd_t*, int port, double* V_reim, double* I_reim);
/* V and I of the most recent step (debug / history recording).  Synchronises the stream. */
int fdtd_read_port_last(fdtd_t*, int port, double* V, double* I);

/* Zero fields, psi, DFT accumulators and the step counter; materials, ports and tables stay. */
int fdtd_reset(fdtd_t*);

/* ---- domain decomposition along z ("decomposing the domain into a number of grids equal to the number
 * of GPUs", guard-cell exchange every step) --------------------------------------------------------------
 * A handle can be one z slab [z0, z1) of a larger grid.  fdtd_set_z_interfaces (before commit) declares which of its z
 * faces are interfaces to a neighbouring slab instead of PEC walls: the halo planes -1 / nz of the padded arrays then
 * hold the neighbour's planes z0-1 / z1, and Ex, Ey on plane 0 of a lo-open slab are ordinary cells.  Such a handle runs
 * the fused step only and advances one step at a time:
 *     fdtd_step_begin   H^{n+1/2} on every plane, E^{n+1} on every plane but plane 0 of a lo-open slab
 *     caller            new Hx, Hy of my plane nz-1  ->  halo plane -1 of the upper neighbour
 *     fdtd_step_end     E^{n+1} on plane 0 of a lo-open slab, then source, probes, DFT of this slab's ports
 *     caller            new Ex, Ey of my plane 0     ->  halo plane nz of the lower neighbour
 * CPML cells on z belong to the first (z-) and last (z+) slab only; a port must lie inside one slab (its I loop reads
 * planes lk0-1 .. lk1).  fdtd_plane returns the device address and byte size of the padded plane k in [-1, nz] of a
 * component in the field set that holds the current state (the new one after fdtd_step_begin); planes of slabs with
 * equal nx, ny have equal size and layout, so an exchange is one contiguous device-to-device copy (NVLink peer copy,
 * ncclSend/ncclRecv).  On a closed handle begin + end is one ordinary step.  Errors: FDTD_ESTATE out of order. */
int fdtd_set_z_interfaces(fdtd_t*, int lo_open, int hi_open);
int fdtd_step_begin(fdtd_t*);
int fdtd_step_end(fdtd_t*);
int fdtd_plane(fdtd_t*, int comp, int k, void** dev_ptr, size_t* bytes);

/* Linked z slabs: the exchange moves INTO the kernels.  Instead of the caller copying planes between
 * fdtd_step_begin and fdtd_step_end, a slab is given the addresses of its neighbours' halo planes once, and from then on
 *   - the fused kernel stores the new Hx, Hy of its top plane also into the upper slab's halo plane -1,
 *   - the kernel that updates E on plane 0 stores the new Ex, Ey also into the lower slab's halo plane nz
 * (plain global stores: NVLink peer stores when the neighbour lives on another GPU -- peer access of another device of
 * this process is enabled by fdtd_z_link; memory of another process must have been opened with CUDA IPC by the caller),
 * and the hand-over is ordered by one 64-bit arrival counter per face in the RECEIVER's memory: the sender posts the step
 * number after its kernel (release at system scope), the receiver's stream waits for it before the kernel that reads the
 * halo (acquire; a bounded spin: FDTD_OPT_Z_SPIN).  Sequence of one step, all of it enqueued by the library:
 *     [wait E(n) from above]  fused kernel  [post H(n+1/2) up]      [wait H(n+1/2) from below]  E on plane 0, source,
 *     probes, DFT  [post E(n+1) down]
 *   fdtd_z_halo(side, planes, flag)   side 0 (z-): where the slab BELOW must put Hx, Hy of its top plane (my halo plane
 *                                     -1), side 1 (z+): where the slab ABOVE must put Ex, Ey of its plane 0 (my halo plane
 *                                     nz): planes[comp + 2*set] for field set 0 and 1 (the step ping-pongs between them;
 *                                     all slabs must step in lockstep from the same reset), flag = my arrival counter.
 *   fdtd_z_link(side, peer_planes, peer_flag)   give this slab the fdtd_z_halo answer of the neighbour on `side`
 *                                     (side 1: the upper slab's side-0 answer; side 0: the lower slab's side-1 answer).
 * Once every open side is linked, fdtd_step(n) works on the slab (and replays captured graphs).  fdtd_step_begin /
 * fdtd_step_end stay available and do the same per half step: slabs that share ONE stream must be advanced that way
 * (all begins, then all ends, in ascending slab order), so that no wait ever precedes its post in stream order; slabs on
 * their own GPUs run fdtd_step(n) concurrently.  A wait that gives up makes the next synchronising read return FDTD_ECUDA.
 * fdtd_reset of a linked slab clears its own halo planes and counters on its own stream only, while the neighbours' kernels
 * store into them: the CALLER must let every linked slab finish (synchronise all their streams, and a barrier between
 * processes) before the first fdtd_reset, and let every reset finish the same way before the next step -- otherwise a late
 * post survives the clear and satisfies the waits of the next run.
 * Errors: FDTD_ESTATE before commit / for a face that is not an interface; FDTD_ECUDA without a peer path. */
int fdtd_z_halo(fdtd_t*, int side, void* planes[4], void** flag);
int fdtd_z_link(fdtd_t*, int side, void* const peer_planes[4], void* peer_flag);

long fdtd_step_count(const fdtd_t*);
/* Number of kernel launches the library has enqueued since commit (graph nodes count individually). */
long fdtd_launch_count(const fdtd_t*);
/* Number of CUDA-graph replays fdtd_step has issued since commit (each covers FDTD_OPT_GRAPH_UNROLL steps). */
long fdtd_graph_replays(const fdtd_t*);
/* Ordinal of the CUDA device the handle was committed on (-1 before commit). */
int fdtd_device(const fdtd_t*);
/* Name of the step implementation in use after commit ("two_pass", "fused"), for reports. */
const char* fdtd_impl_name(const fdtd_t*);
/* z chunk length of the fused step in use after commit (0 for the two-pass step), for reports.  With
 * FDTD_OPT_STEP_IMPL = 0 or FDTD_OPT_FUSED_KZ = 0, fdtd_commit times the candidates on the committed all-zero state
 * (two-pass and fused with 12..48 planes per chunk) and keeps the fastest; the state is left exactly as committed. */
int fdtd_fused_kz(const fdtd_t*);
/* Tile of the fused step in use after commit, numbered as FDTD_OPT_FUSED_TILE (1 or 2; 0 when another step implementation
 * is in use), for reports. */
int fdtd_fused_tile(const fdtd_t*);
/* FDTD_OPT_STEP_IMPL = 4 (in use after commit): the box [box[0], box[1]) x [box[2], box[3]) x [box[4], box[5]) of cells that one
 * kernel advances two steps per pass; every other cell belongs to the shell that the one-step kernels advance (reports:
 * the bytes one launch of the two-step kernel must move are counted over this box).  FDTD_ESTATE when another step
 * implementation is in use. */
int fdtd_two_step_box(const fdtd_t*, int box[6]);
const char* fdtd_last_error(const fdtd_t*);
void fdtd_destroy(fdtd_t*);

/* ---- port probes for callers that cannot allocate device memory ------------------------------------------------------------
 * V and I of Eq. 4 (reading R7; the formulas stand above fdtd_port) of `nports` ports, from field arrays the
 * caller already holds, without a handle and without a workspace.  Meant for code that has no way to obtain device memory when
 * it wants a probe: a monitor looking at a run in flight (an allocation would synchronise the GPU under the time stepping), a
 * plug-in whose host program took the whole GPU for its own pool at start-up (an allocation fails there), a hook that runs
 * where allocator calls are forbidden.  The reduction is spread over several thread blocks per port and needs a little memory
 * for the hand-over between them; this entry point keeps it in a fixed array inside the library image
 * (FDTD_NOALLOC_SCRATCH_BYTES per GPU, resident on every GPU that loads the library until the process exits) and calls no
 * allocation routine of any kind.
 *   Ez, Hy, Hz   DEVICE arrays of nx*ny*nz elements of `precision` (FDTD_F32 | FDTD_F64), index i + nx*(j + ny*k), all on one
 *                GPU; read only.  E.g. what fdtd_read_fields wrote, or another solver's fields.
 *   ports        HOST array; only ip, v* and l* are read (the source part is ignored).  Same range rules as fdtd_add_port.
 *   VI           DEVICE array of 2*nports doubles on the same GPU: VI[2p] = V, VI[2p+1] = I of port p.  Written by the kernel;
 *                valid once the stream has reached that point.  The reduction is carried out in fp64 whatever the precision.
 *   cuda_stream  a cudaStream_t of that GPU as void* (NULL = the legacy default stream).  One memset and one kernel are
 *                enqueued; nothing is synchronised.
 *   errbuf       optional HOST buffer for a message on failure (there is no handle to ask); may be NULL.
 * Limits and sharing -- all of them consequences of the one built-in array:
 *   - at most FDTD_NOALLOC_MAX_PORTS ports per call; a longer list returns FDTD_ERANGE and enqueues nothing (split it);
 *   - every call on a GPU uses the same array, which still holds the previous call's contents; the call clears the arrival
 *     counters (the only part that must start at zero) on the stream before its kernel;
 *   - calls whose kernels may run at the same time on one GPU (two streams, two threads) race on that array and give wrong
 *     answers; calls on one stream are ordered and fine, and different GPUs have different copies;
 *   - the first call on each GPU looks up where that GPU's copy of the array lives (cudaGetSymbolAddress, with that GPU made
 *     current) and caches the address: make this first call before any stream capture begins.
 * Returns FDTD_OK, FDTD_EINVAL (bad precision / sizes / null or non-device pointers / arrays on different GPUs), FDTD_ERANGE
 * (too many ports, a port outside the grid, ny*nz above 2^31-1) or FDTD_ECUDA.  The caller's current device is restored. */
enum { FDTD_NOALLOC_MAX_PORTS = 16, FDTD_NOALLOC_MAX_BLOCKS = 64,
       FDTD_NOALLOC_SCRATCH_BYTES = 2 * 8 * FDTD_NOALLOC_MAX_BLOCKS * FDTD_NOALLOC_MAX_PORTS + 256 };
int fdtd_port_probe_noalloc(const void* Ez, const void* Hy, const void* Hz, int precision, int nx, int ny, int nz,
                            double dy, double dz, const fdtd_port* ports, int nports, double* VI, void* cuda_stream,
                            char* errbuf, size_t errbuf_len);

#ifdef __cplusplus
}
#endif
#endif /* FDTD_B200_H */
