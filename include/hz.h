/* hz.h -- C ABI of the B200-native HORIZON GRMHD update (libhz.so).
 *
 * What the library does: it advances ideal GRMHD in 3+1 conservative form on a uniform Cartesian
 * mesh in a fixed, given spacetime by method-of-lines Runge-Kutta substeps.  One substep is the
 * pipeline of PAPER.md:74-80 (section 2.2): reconstruct the primitives at the faces, evaluate
 * left/right fluxes and maximal wave speeds, take an approximate (HLLE) Riemann flux, difference the
 * fluxes and add the local geometric source terms of PAPER.md:54 (eq. 2), combine the Runge-Kutta
 * stage, recover the primitives by Newton-Raphson and refill the ghost zones.  The named
 * ingredients are those of PAPER.md:128 (section 3.2): HLLE, TVD reconstruction with the MC limiter,
 * third-order Runge-Kutta, Newton-Raphson primitive recovery, hyperbolic divergence cleaning.  Every
 * discrete formula the paper does not print is a reading listed in DESIGN.md (R1-R22).
 *
 * Every step of that path runs in hand-written CUDA kernels for sm_100a, in fp64 or fp32 (one dtype
 * per context).  There is NO CPU fallback: without a CUDA device every compute entry point returns
 * HZ_ECUDA.
 *
 * Conventions
 *   Layout    Every field array is INTERIOR-ONLY, nx*ny*nz elements per plane, x fastest
 *             (PAPER.md:152), planes concatenated.  Element type = the context dtype
 *             (HZ_F32: float, HZ_F64: double).  The library pads, adds ghost zones and fills
 *             them itself.
 *   Pointers  Every `const void*` / `void*` field argument may be a HOST pointer (pageable or
 *             pinned) or a DEVICE pointer; the library resolves which with
 *             cudaPointerGetAttributes and copies.  The caller owns these buffers before and
 *             after the call; the library keeps no reference to them.
 *   Stream    All device work of a context is enqueued on its stream (default: the legacy default
 *             stream; hz_set_stream changes it).  hz_step / hz_substeps are ASYNCHRONOUS: they
 *             return once the work is enqueued.  hz_set_*, hz_get_* and hz_diagnostics
 *             synchronise the stream before returning.
 *   Errors    Every call returns an int: HZ_OK (0) or a negative code.  No exception crosses
 *             the ABI and the library never exits the process.
 *   Units     G = c = 1; B^i is the Eulerian-observer magnetic field with 1/sqrt(4 pi) absorbed
 *             (b^2 adds to rho h without a 4 pi).  Velocities at the boundary are the Eulerian
 *             3-velocity v^i (contravariant); internally the library stores W v^i
 *             (footnote 3).
 */
#ifndef HZ_H
#define HZ_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct hz_ctx hz_ctx; /* opaque; created by hz_create, freed by hz_destroy */

/* HZ_F32_F64: the paper's mixed mode: fields stored and face fluxes computed in
 * fp32 (arrays at the boundary are float, as for HZ_F32); flux difference, Runge-Kutta combine and
 * primitive recovery in fp64. */
enum { HZ_F32 = 0, HZ_F64 = 1, HZ_F32_F64 = 2 };
/* Per axis.  The three EXTERNAL codes are for the z axis only (slab decomposition across GPUs,
 * PAPER.md:176-178): the ghost planes of an external side are not filled by the library's boundary
 * rule but supplied by the caller through hz_halo_unpack.  HZ_BC_EXTERNAL: both sides external;
 * HZ_BC_EXTERNAL_OUTFLOW: low side external, high side outflow; HZ_BC_OUTFLOW_EXTERNAL: the reverse. */
enum { HZ_BC_PERIODIC = 0, HZ_BC_OUTFLOW = 1, HZ_BC_EXTERNAL = 2, HZ_BC_EXTERNAL_OUTFLOW = 3,
       HZ_BC_OUTFLOW_EXTERNAL = 4 };
enum { HZ_OK = 0, HZ_EINVAL = -1, HZ_ENOMEM = -2, HZ_ECUDA = -3, HZ_ESTATE = -4,
       HZ_ELIMIT = -5 /* a size beyond the fixed maximum of hz_sum_fields_noalloc */ };

/* Uniform Cartesian mesh.  An axis with one cell is inactive: no ghost zones, no
 * sweep, no derivative along it (two-dimensional meshes). */
typedef struct { int nx, ny, nz; double dx, dy, dz; int bc[3]; } hz_grid;

typedef struct {
  double gamma_ad;        /* ideal-gas adiabatic index Gamma (> 1)                              */
  double rho_atm, p_atm;  /* atmosphere values; also the floors of the face states              */
  double atm_tol;         /* a cell is reset to atmosphere if rho < rho_atm*(1+atm_tol)         */
  int    cleaning;        /* 0: psi frozen at 0; 1: hyperbolic divergence cleaning */
  double kappa;           /* cleaning damping rate                                              */
  int    c2p_maxit;       /* Newton iteration cap of the primitive recovery                     */
  double c2p_tol;         /* converged when |dZ| <= c2p_tol*Z; <= 0 selects the dtype default   */
                          /* (1e-13 for HZ_F64, 1e-6 for HZ_F32, 1e-10 for the fp64 recovery of */
                          /* HZ_F32_F64).  HZ_F32 measures the step against Z + B^2 (the round- */
                          /* off of the residual is eps*(Z + B^2)) and also accepts a step that  */
                          /* has stopped shrinking below 64 eps of that scale (counted in        */
                          /* hz_diag.c2p_stalled); no other acceptance exists                    */
  int    c2p_scheme;      /* 0: Newton on Z = rho h W^2; 1: Newton on the two unknowns (Z, v^2),  */
                          /* the paper's second recovery scheme.  Same root.       */
  int    energy_var;      /* 0: the energy slot of U is sqrt(gamma) tau (north_star); 1: the paper's */
                          /* own variable -sqrt(-g) T^t_t = sqrt(gamma)[alpha(tau+D) - beta^j S_j]   */
                          /* (PAPER.md:54, 60), which has no source on a fixed metric; hz_get_conserved */
                          /* and hz_diag.sumTau then carry that variable.                            */
  int    recon;           /* reconstruction: 0 TVD with the MC limiter (2 ghost layers), */
                          /* 1 PPM (3 ghost layers; an active axis then needs at least 3 cells)       */
} hz_params;

/* Global reductions, all accumulated in fp64. */
typedef struct {
  double sumD, sumSx, sumSy, sumSz, sumTau;  /* sum over interior cells of sqrt(gamma)*(..)*dx*dy*dz */
  double sumBx, sumBy, sumBz, sumPsi;
  double divB_max, divB_L1;                  /* centred div(sqrt(gamma) B)/sqrt(gamma): max, mean |.| */
  double max_speed_over_dx;                  /* max over cells, axes of max(|lam+|,|lam-|)/dx_d       */
  long long c2p_fail, atm_reset, p_floor;    /* cumulative since hz_set_primitives                    */
  int c2p_maxit_seen;
  long long c2p_stalled;                     /* HZ_F32 only: recoveries accepted by the round-off rule */
                                             /* of c2p_tol below (not failures; cumulative)            */
} hz_diag;

/* Fill *p with the defaults: Gamma = 4/3, atmosphere 1e-12 / 1e-14, atm_tol 1e-3, cleaning on,
 * kappa = 1, 30 Newton iterations, c2p_tol = 0 (dtype default), c2p_scheme = 0, energy_var = 0, recon = 0.  HZ_EINVAL if p is NULL. */
int hz_default_params(hz_params* p);

/* Bytes of device memory one context of this grid and dtype needs (all resident fields: metric,
 * two primitive sets, conserved, conserved at the step start, staging and reduction scratch).
 * HZ_EINVAL on a bad grid or dtype.  Needs no GPU. */
int hz_state_bytes(const hz_grid* grid, int dtype, size_t* bytes);
/* The same for the layout hz_create builds with `params` (NULL = defaults): 2 ghost layers with the MC
 * reconstruction, 3 with PPM; hz_state_bytes above is the larger of the two, enough for either. */
int hz_state_bytes_for(const hz_grid* grid, int dtype, const hz_params* params, size_t* bytes);

/* Create a context.  `device_buffer` is either NULL (the library allocates hz_state_bytes with
 * cudaMalloc and frees it in hz_destroy) or a caller-owned DEVICE buffer of at least hz_state_bytes
 * bytes (hz_state_bytes_for(.., params, ..) suffices), 256-byte aligned (e.g. a torch.uint8 tensor's data_ptr()), which
 * must outlive the context.
 * `params` may be NULL (defaults).  Errors: HZ_EINVAL (bad grid: n < 1, 1 < n < 2 along an axis,
 * spacing <= 0, unknown bc or dtype, Gamma <= 1, maxit < 1), HZ_ECUDA (no device / CUDA failure),
 * HZ_ENOMEM. */
int hz_create(const hz_grid* grid, int dtype, const hz_params* params, void* device_buffer, hz_ctx** out);
int hz_destroy(hz_ctx* ctx);

/* Use `cuda_stream` (a cudaStream_t, e.g. torch.cuda.current_stream().cuda_stream; NULL = default
 * stream) for all later work of this context. */
int hz_set_stream(hz_ctx* ctx, void* cuda_stream);

/* Fixed spacetime: lapse `alpha` (1 plane), shift `beta3` (beta^x, beta^y, beta^z:
 * 3 planes), spatial metric `gamma6` (xx, xy, xz, yy, yz, zz: 6 planes).  Ghost zones are filled by
 * periodic wrap or by copying the nearest interior cell (outflow axes).  HZ_EINVAL if any value is
 * non-finite, alpha <= 0 or gamma_ij is not positive definite.  Invalidates the primitives. */
int hz_set_metric(hz_ctx* ctx, const void* alpha, const void* beta3, const void* gamma6);

/* Initial data in primitive variables: `prim8` = rho, v^x, v^y, v^z, p, B^x, B^y, B^z
 * (8 planes).  Runs prim->cons and the ghost fill; sets psi = 0, the Runge-Kutta stage
 * to 0 and the counters of hz_diag to 0.  HZ_ESTATE before hz_set_metric; HZ_EINVAL if a value is
 * non-finite, rho <= 0, p < 0 or v^2 >= 1. */
int hz_set_primitives(hz_ctx* ctx, const void* prim8);

/* Advance n full third-order Runge-Kutta steps (= 3n substeps) with the fixed step dt
 * (PAPER.md:128, 238).  Asynchronous.  HZ_ESTATE before metric and primitives are set or in the
 * middle of a step (after hz_substeps with a count not divisible by 3); HZ_EINVAL if dt <= 0, n < 0.
 * Failed primitive recoveries are not errors: the cell is reset to atmosphere and counted.
 * With n >= 2 the launches of two consecutive steps (six substeps, after which the double buffers are back in
 * their roles) are captured once into a CUDA graph and replayed n / 2 times, ordered behind and before the
 * context stream by events; an odd last step and everything hz_substeps does are plain launches.  The results are
 * the same bit for bit; the environment variable HZ_NO_GRAPH=1 (read at hz_create) turns the replay off. */
int hz_step(hz_ctx* ctx, double dt, int n);
/* Advance `nsub` Runge-Kutta substeps, continuing from the current stage.  Asynchronous. */
int hz_substeps(hz_ctx* ctx, double dt, int nsub);

/* Current primitives in the layout of hz_set_primitives (v^i = W v^i / W), the cleaning scalar psi
 * (1 plane) and the densitised conserved variables sqrt(gamma)*(D, S_x, S_y, S_z, tau, B^x, B^y,
 * B^z, psi) (9 planes). */
int hz_get_primitives(hz_ctx* ctx, void* prim8);
int hz_get_psi(hz_ctx* ctx, void* psi);
int hz_get_conserved(hz_ctx* ctx, void* cons9);

/* Global reductions over the current state.  Synchronises the stream. */
int hz_diagnostics(hz_ctx* ctx, hz_diag* out);

/* Ghost-zone exchange of a slab decomposition along z (pack kernel, transfer, unpack
 * kernel, every substep; here the transfer is device-to-device and the caller's: NCCL send/recv over
 * NVLink between processes, or a plain copy between contexts of one process).  `which` selects the
 * primitives (9 fields) or the metric (10 fields); `side` 0 = low z, 1 = high z.
 * hz_halo_pack copies the NG interior planes next to that side (NG = 2 with MC, 3 with PPM) -- whole padded planes, so the x and y
 * ghost columns travel too -- into `device_buf` (hz_halo_bytes bytes, DEVICE memory, context dtype);
 * hz_halo_unpack writes such a buffer into the ghost planes of that side.  A slab's low-side buffer
 * goes to the high-side ghosts of the slab below it and vice versa.  Both are asynchronous on the context
 * stream.  Call order per substep: hz_substeps(dt, 1) on every slab, pack, transfer, unpack; and once after
 * hz_set_metric (metric) and after hz_set_primitives (primitives).  The library keeps track: hz_set_metric,
 * hz_set_primitives and every substep invalidate the ghost planes of the external sides they outdate, and
 * hz_substeps / hz_step return HZ_ESTATE instead of advancing a slab whose external ghost planes (metric or
 * primitives) have not been supplied since.  HZ_EINVAL if z is inactive or the buffer is not device memory;
 * HZ_ESTATE before the fields are set. */
enum { HZ_HALO_PRIM = 0, HZ_HALO_METRIC = 1 };
int hz_halo_bytes(const hz_ctx* ctx, int which, size_t* bytes);
int hz_halo_pack(hz_ctx* ctx, int which, int side, void* device_buf);
int hz_halo_unpack(hz_ctx* ctx, int which, int side, const void* device_buf);

/* The exchange of the primitives FUSED INTO THE SUBSTEP KERNEL (PAPER.md:176-178 exchanges the ghost zones after
 * every substep with a pack kernel, two copies through the host, MPI and an unpack kernel; PAPER.md:278 names that
 * synchronisation as the possible limit of the scaling).  Where the neighbour's primitive buffers are addressable
 * from this device -- another context on the same GPU, a peer GPU of this process (cudaDeviceEnablePeerAccess), or
 * another process's buffer opened through CUDA IPC -- hz_peer_attach hands them to the context, and from then on
 * every substep stores the cells within NG planes of that cut, and their x / y ghost images, straight into the
 * neighbour's ghost planes (over NVLink for a peer GPU) while it writes its own primitives: no pack kernel, no
 * transfer, no unpack kernel, and hz_halo_pack / hz_halo_unpack of the primitives are needed only once, after
 * hz_set_primitives.  (The metric's ghost planes are exchanged once with hz_halo_pack / hz_halo_unpack as before.)
 *   hz_prim_buffers  the DEVICE addresses of this context's two primitive sets (9 fields each, `field_stride`
 *                    elements apart, padded layout) -- what the neighbour passes to hz_peer_attach.  They are part
 *                    of the state buffer and live as long as the context.
 *   hz_peer_attach   side 0 = the neighbour below (low z), 1 = above; peer_P0 / peer_P1 / peer_field_stride: the
 *                    neighbour's hz_prim_buffers; peer_nz: its interior planes.  The neighbour must have the same
 *                    nx, ny, dtype, reconstruction and boundary kinds in x and y.  HZ_EINVAL if that side is not
 *                    external, a pointer is not device memory, or the context does not run the default
 *                    configuration (cleaning on, energy_var 0: the only kernels compiled with peer stores).
 *   hz_peer_detach   back to hz_halo_pack / hz_halo_unpack on that side.
 * Contract: attach MUTUALLY (each of two neighbours attaches the other) and advance the slabs in LOCKSTEP -- every
 * slab takes substep s before any takes s + 1, and a slab's substep s + 1 is ordered behind its neighbours' substep s
 * on the device (one stream, an event, or a barrier between processes); the library then regards the ghost planes
 * of an attached side as supplied after each substep and does not return HZ_ESTATE for them.  Nothing is allocated
 * and the library keeps only the three pointers; the caller keeps the neighbour's buffers alive. */
int hz_prim_buffers(hz_ctx* ctx, void** P0, void** P1, long long* field_stride);
int hz_peer_attach(hz_ctx* ctx, int side, void* peer_P0, void* peer_P1, long long peer_field_stride, int peer_nz);
int hz_peer_detach(hz_ctx* ctx, int side);

/* Number of kernels this context has launched since hz_create (bench.py's gpu_launches). */
long long hz_launch_count(const hz_ctx* ctx);

/* Measured throughput of the plain FMA pipe in `dtype` (HZ_F32 or HZ_F64), TFLOP/s with FMA = 2 flops:
 * a kernel of nothing but independent FMAs on every SM, best of three timed launches on the default stream.
 * It is the measured counterpart of the derived ALU peak the roofline is quoted against.
 * Needs no context.  HZ_ECUDA without a device. */
int hz_fma_peak(int dtype, double* tflops);

/* Per-kernel device timing of the substep kernels, for the roofline report (PAPER.md:190-194 times
 * the main loop only).  hz_profile(ctx, 1) brackets every later substep kernel launch with CUDA
 * events on the context stream; hz_profile_read synchronises, adds up the elapsed milliseconds and
 * the launch counts per kernel kind (arrays of HZ_NKERNELS entries, kind k named hz_kernel_name(k))
 * and clears the record.  At most 16384 launches are kept between reads; later ones are not timed. */
enum { HZ_NKERNELS = 2 };
int hz_profile(hz_ctx* ctx, int enable);
int hz_profile_read(hz_ctx* ctx, double* ms, long long* launches);
const char* hz_kernel_name(int kind);

/* ---- the one entry point that allocates NOTHING (csrc/hz_noalloc.cu) -------------------------------------
 * For callers that cannot call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that
 * forbid it.  A variant of the library's global reduction (hz_diagnostics) that needs no
 * context: the sums over `ncell` cells of `nfields` fields, accumulated in fp64 in a fixed order (deterministic).
 *   fields_dev  DEVICE memory, nfields planes of ncell elements each, plane f at element offset f*ncell
 *               (the layout hz_get_conserved writes), element type float (HZ_F32) or double (HZ_F64)
 *   sums_dev    DEVICE memory, nfields doubles: sums_dev[f] = sum of plane f.  (Multiply by dx*dy*dz for the
 *               volume sums hz_diagnostics reports.)
 *   cuda_stream a cudaStream_t (NULL = default stream); the call is ASYNCHRONOUS, two kernels on that stream
 * The block partials live in a file-scope `static __device__` array of fixed size --
 * HZ_NOALLOC_MAX_BLOCKS x HZ_NOALLOC_MAX_FIELDS doubles = 151 552 bytes (148 KiB) -- which every GPU that loads
 * the library holds until the process exits.  Limits: nfields <= HZ_NOALLOC_MAX_FIELDS (16) and
 * ncell <= HZ_NOALLOC_MAX_CELLS (2^31 cells per field); beyond them the call returns HZ_ELIMIT and does nothing.
 * The call itself performs no cudaMalloc, cudaFree or allocating library call.  hz_noalloc_setup looks up the
 * array's device address for the CURRENT device (cudaGetSymbolAddress; once per device; no allocation, no
 * launch); hz_sum_fields_noalloc does the same on its first call on a device, so call hz_noalloc_setup first
 * where even that look-up is unwelcome (before a stream capture begins).
 * Every call on a device shares the one array, which keeps the last call's contents; nothing in it has to start
 * at zero (every row a call reads it has written first).  Calls that OVERLAP on one GPU -- different streams or
 * host threads without ordering between them -- race on the array and return wrong sums: serialise them.
 * Errors: HZ_EINVAL (NULL or non-device pointer, nfields < 1, ncell < 1, dtype not HZ_F32 / HZ_F64; the mixed
 * mode stores floats: pass HZ_F32), HZ_ELIMIT, HZ_ECUDA. */
#define HZ_NOALLOC_MAX_BLOCKS 1184
#define HZ_NOALLOC_MAX_FIELDS 16
#define HZ_NOALLOC_MAX_CELLS (1LL << 31)
int hz_noalloc_setup(void);
int hz_sum_fields_noalloc(const void* fields_dev, int nfields, long long ncell, int dtype, double* sums_dev,
                          void* cuda_stream);

const char* hz_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif
