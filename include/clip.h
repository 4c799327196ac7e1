/*
 * clip.h -- C ABI of libclip: the per-timestep update of the two D3Q19 population sets (Allen-Cahn `g`,
 * velocity/pressure `f`) of the conservative phase-field lattice Boltzmann method of arxiv 2505.12205,
 * hand-written CUDA for sm_100a (B200).  Citations are PAPER.md line numbers / equation numbers.
 *
 * Problem statement (PAPER.md:341 Fig. 4a, :541 Alg. 3 "Ensure"): initial phi and u in; after n time steps
 * phi, p, u out.  One step = collision (Alg. 1, :351-429) -> streaming (Alg. 2, :432-459) -> boundary conditions
 * (App. B, :963-1129) -> macroscopic variables (Alg. 3, :461-541).
 *
 * Conventions
 *   - Lattice units dx = dt = c = 1, c_s^2 = 1/3 (:172, :193).  Paper tau: nu = tau/3 (Eq. 23), rate 1/(tau+1/2).
 *   - Field layout: scalar fields [nz][ny][nx] with x fastest (Fig. 4b, :343); vectors SoA [3][nz][ny][nx].
 *   - Every `d_*` pointer is a DEVICE pointer; element type is float (precision 32) or double (precision 64),
 *     for the workspace and for all user I/O alike.  Pointers must be aligned to 16 bytes.
 *   - Ownership: the caller owns every device buffer, including the workspace, and keeps the workspace alive
 *     until clip_destroy.  The library never allocates device memory.  clip_init / clip_get read / write their
 *     arguments asynchronously on the handle's stream and do not retain them.
 *   - The handle is a host heap object owned by the library.  One handle = one stream; not thread-safe.
 *   - Errors: every int-returning call returns CLIP_OK (0) or a negative code; no exceptions, no aborts, no
 *     host synchronisation inside clip_step.  Text via clip_last_error.
 */
#ifndef CLIP_H_
#define CLIP_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { CLIP_OK = 0, CLIP_EINVAL = -1, CLIP_ENOMEM = -2, CLIP_ESTATE = -3, CLIP_ECUDA = -4 };

/* Boundary type of one lattice face.  PERIODIC: App. B.1 (:971-1003).  WALL: halfway bounce-back, App. B.3
 * (:1028-1038).  INLET: velocity inlet, App. B.4 (:1042-1088), only on the -z face.  OUTLET: convective outlet,
 * App. B.5 (:1094-1129), only on the +z face.  FREESLIP: specular reflection half a cell outside the last node, App. B.2
 * (B.8-B.9, :1017-1026): zero normal velocity, free tangential velocity; where a link also crosses a WALL face the
 * bounce-back wins.  The phi stencils (Eq. 40) take the mirror value behind WALL, FREESLIP, INLET and OUTLET faces. */
enum { CLIP_BC_PERIODIC = 0, CLIP_BC_WALL = 1, CLIP_BC_INLET = 2, CLIP_BC_OUTLET = 3, CLIP_BC_FREESLIP = 4, CLIP_BC_HALO = 5 };
/* CLIP_BC_HALO (z faces only): the cut face of a z slab of a larger lattice.  The first / last plane of such a
 * lattice is a GHOST plane -- an image of the neighbouring slab's outermost owned plane, refreshed by clip_halo_unpack after every
 * step -- and clip_step advances the owned planes only.  See clip_halo_pack. */

/* Hydrodynamic collision operator: weighted MRT (the paper's choice for 3-D, :849) or BGK. */
enum { CLIP_COLL_WMRT = 0, CLIP_COLL_BGK = 1 };

typedef struct clip_params {
  int precision;           /* 32 or 64: element type of every device array incl. user I/O */
  double rho_h, rho_l;     /* densities of the phi=1 (heavy) and phi=0 (light) fluid, Eq. 39 (:301) */
  double tau_h, tau_l;     /* paper relaxation times, nu = tau/3, Eq. 23-24 (:209-213) */
  double sigma, W, M;      /* surface tension, interface width xi, mobility: Eq. 12 (:154), 34 (:277), 37 (:293) */
  double g[3], rho_ref;    /* body force F_b = (rho - rho_ref) g  (Eq. 58 :825; rho_ref = 0 gives rho g, :649) */
  int bc[6];               /* faces -x,+x,-y,+y,-z,+z : CLIP_BC_* ; PERIODIC faces must come in pairs */
  double inlet_u[3];       /* plug inflow velocity u_in, B.12 (:1048) */
  double inlet_phi;        /* phi_in, B.16 (:1069) */
  double inlet_c[2];       /* nozzle disc centre (x, y) in node coordinates */
  double inlet_r;          /* nozzle radius; nodes of the -z face outside the disc are WALL */
  int outlet_u_mode;       /* characteristic outlet velocity U of B.22 (:1104), built on the normal velocity of layer N-1:
                              0 = U_local (per column), 1 = U_ave (mean over the layer), 2 = U_max */
  int visc_interp;         /* 0 = linear tau, Eq. 24 (paper, Alg. 1); 1 = harmonic (1/tau linear in phi; non-paper);
                              2 = linear dynamic viscosity, Eq. 25 (:219): mu = rho tau / 3, tau = 3 mu(phi) / rho(phi) */
  int collision;           /* CLIP_COLL_WMRT (0, default): Eq. 27-28 + F_mu of Eq. 30; CLIP_COLL_BGK (1): Eq. 26 + F_mu of Eq. 29 */
  int phase_only;          /* 0 (default): full two-phase flow.  1: only the phase-field equation (Eq. 33) is advanced and
                              u is prescribed by the caller (clip_set_u) -- the set-up of the interface-in-shear-flow test,
                              PAPER.md:675-713 (Sec. 5.4); f stays 0, p is returned as 0 */
  int outlet_clamp;        /* lambda of B.25 (:1115-1117): 0 (default) = U dt/dy exactly as printed; 1 = max(0, U).  B.21 is an
                              OUTFLOW condition: for U < 0 the implicit upwind form B.23-B.25 multiplies chi(N) - chi(N-1) by
                              1/(1 + lambda) > 1 every step (reading R12); with the clamp such columns keep
                              chi(N, t+dt) = chi(N, t).  Lattices whose outlet sees backflow (the jet into quiescent gas) want 1 */
  int outlet_u_time;       /* which velocity enters B.22 (the paper says both, :1107 and :1117; reading R12):
                              0 (default) = the stored macroscopic u_z(x,y,N-1,t) of the previous time step; 1 = the first moment
                              sum_a e_az f_a(x,y,N-1,t+dt) of the post-stream populations (not in phase_only mode) */
  int path;                /* kernel path of clip_step (not part of the method; all paths compute the same step): 0 = automatic
                              (see clip_step), 1 = generic kernels only, 2 = never k_fused (pair kernels where the lattice admits
                              them), 3 = k_fused wherever the lattice admits it, 4 = k_fused_tma (k_fused fed by bulk-async copies through
                              shared memory; x / y faces PERIODIC) where admitted, else as 3; 5 = the same with only the g populations staged (experiments,
                              profiles/r02_experiments.md).  The slabs of one lattice must agree on whether
                              phi(t+1) is kept in a second buffer */
  int tile_ty, tile_chunks; /* k_fused tiling (tests / tuning; 0 = automatic): lattice rows per tile (4, 8 or 16, must divide ny) and
                              number of equal chunks along z (1 .. min(nz, 256)); they enter clip_workspace_bytes */
  int runtime_nx;          /* 1 = take the runtime-nx instantiation of the pair kernels even where nx has its own (tests) */
  int lattice;             /* velocity set: 0 (default) = D3Q19, Eq. 14-15 (:169-176); 1 = D2Q9, the lattice of the paper's 2-D benchmarks
                              (:568): nz must be 1, the z faces PERIODIC, the x / y faces PERIODIC, WALL or FREESLIP; u_z is returned as
                              given to clip_init (0).  Pair-per-thread kernels k_phi9p + k_step9p where nx is even, else the thread-per-node
                              kernels k_phi9 + k_step9; path = 3 takes the single-pass kernels k_fused9 + k_fix9 where nx % 64 == 0 (an option:
                              measured slower than the pair kernels, profiles/r02_experiments.md 4f) */
  int cluster_y;           /* k_fused, tuning / tests: y-adjacent tiles per thread-block cluster, whose shared tile surfaces are completed
                              through distributed shared memory instead of the partial-sum buffer.  0 = automatic (fp32: 4 at nx = 128,
                              2 at nx = 192, the lattices with 64- / 96-thread blocks, where it is measured to pay; else none),
                              1 = none, 2, 4 or 8 = that many where the number of y tiles is a multiple (else none).  Same results bit
                              for bit */
} clip_params;

typedef struct clip_handle clip_t;

/* Bytes of device workspace clip_create needs for this lattice; 0 if the arguments are invalid. */
size_t clip_workspace_bytes(int nx, int ny, int nz, const clip_params* params);

/* Validate, carve `d_workspace` (device, >= clip_workspace_bytes, 256-byte aligned) and bind to `cuda_stream`
 * (a cudaStream_t / CUstream passed as void*; NULL = default stream).  Copies *params.  Host only apart from
 * one small asynchronous upload (the inlet mask).  On failure *out = NULL and the reason is available from
 * clip_last_error(NULL). */
int clip_create(clip_t** out, int nx, int ny, int nz, const clip_params* params, void* d_workspace, size_t bytes,
                void* cuda_stream);

/* Set t = 0 from phi0 [nz][ny][nx] and u0 [3][nz][ny][nx] (device): p* = 0, populations at the barred
 * equilibria g = phi Gamma - F^phi/2, f = (Gamma - w) - F_a/2 with F = F_s + F_b (Eq. 16-19, 34-36; the paper
 * only says "Initialization", :341 -- DESIGN.md reading R8). */
int clip_init(clip_t* h, const void* d_phi0, const void* d_u0);

/* Advance n >= 0 time steps (Eq. 13, 33 with all of App. B); asynchronous on the stream.
 * Which kernels run is decided per lattice at clip_create: k_fused + k_fix on wide lattices, k_phi2 + k_step2
 * on the other lattices with even nx, the generic k_phi + k_step otherwise (and on the planes next to an INLET / OUTLET face).
 * All paths compute the same step; they agree to round-off, and each is deterministic: clip_step(a); clip_step(b) equals
 * clip_step(a + b) bit for bit.  clip_params.path / tile_ty / tile_chunks / runtime_nx override the choice (tests, tuning); the
 * library reads nothing from the environment.  On lattices of up to 4 M nodes (launch-bound), n >= 32 and a stream that can be captured
 * (not the legacy default stream), the steps are replayed 16 at a time from a CUDA graph the handle captures once.
 * Capture by the CALLER: called while the handle's stream is being captured, clip_step records its launches into the caller's graph
 * and starts no capture of its own.  Such a graph may be replayed any number of times if it holds an EVEN number of steps (the two
 * population buffers and, on the k_fused path, the two phi buffers swap roles every step) and the handle took at least one step
 * outside the capture since clip_init (the k_fused path's one-off phi pre-pass is then behind it); no other call on the handle
 * goes into the same graph, phase_only lattices (clip_set_u between steps) excepted from this use.  The handle's counters
 * (clip_launch_count) advance at capture, not at replay. */
int clip_step(clip_t* h, int n);

/* phase_only mode: prescribe the velocity field u [3][nz][ny][nx] (device) that the following collisions use; the
 * buffer is copied asynchronously on the stream and not retained.  Because the populations are stored post-collision,
 * the field passed before clip_step(h, 1) at time t must be u(t+1) (clip_init takes u(0)).  CLIP_ESTATE outside
 * phase_only mode or before clip_init. */
int clip_set_u(clip_t* h, const void* d_u);

/* Write phi, the physical pressure p = p* rho c_s^2 (:189) and u at the current time into caller buffers
 * (device; any may be NULL); asynchronous on the stream. */
int clip_get(clip_t* h, void* d_phi, void* d_p, void* d_u);

/* z-slab decomposition over several GPUs: one process per GPU holds a slab of consecutive z planes as an ordinary
 * clip_t whose cut faces are CLIP_BC_HALO (one ghost plane per cut).  Streaming pulls every population from at most one plane away
 * (Eq. 13, 33; Alg. 2 :432-459) and the stencils of Eq. 40 (:307-309) read phi one plane away, so what an owned plane needs from
 * the ghost plane next to it is: the 5 f+ and 5 g+ populations that move towards it, and phi of the next collision there.  Per
 * step and per cut each side sends ONE record of 12 words per face node (clip_halo_bytes bytes, layout [12][ny][nx]):
 *   0-4 f+_a, 5-9 g+_a of its boundary plane B for the five directions a that point at the neighbour;
 *   10  the part of phi_B(t+1) = sum_a g+_a(x - e_a, t) that comes from its own side (links bounced at an x / y wall included);
 *   11  C: what B sends into the neighbour's boundary plane, sum over those five a of g+_a(x - e_a) (in-plane faces applied).
 * The receiver completes both boundary planes by additions: phi_ghost = received[10] + (its own C, just sent), and, on the
 * k_fused path (whose on-chip scatter cannot see the ghost's populations), phi_B += received[11]; the ghost plane's ten
 * populations are stored as they are.  phi is therefore summed in a different order than on the undivided lattice: the slabs
 * reproduce it to round-off, not bit for bit.
 *   clip_halo_pack(h, d_lo, d_hi)    writes the records of the -z / +z HALO face into d_lo / d_hi (device, 16-byte aligned,
 *                                    clip_halo_bytes(h) each; NULL for a face that is not HALO).  One launch.
 *   clip_halo_unpack(h, d_recv_lo, d_recv_hi, d_sent_lo, d_sent_hi)
 *                                    d_recv_lo = the record the slab BELOW packed for its +z face, d_recv_hi = the record the slab
 *                                    above packed for its -z face, d_sent_* = what this handle packed at the same time.  One launch.
 * Both are asynchronous on the handle's stream; the transfer between GPUs is the caller's (paper_2505_12205_b200/slab.py: NCCL
 * send / recv between z neighbours).  Protocol: clip_init; pack, exchange, unpack; then per step: clip_step(h, 1); pack, exchange,
 * unpack.  A physical z face of the whole lattice (WALL, FREESLIP, INLET, OUTLET) belongs to the first / last slab.  The outlet's
 * U_ave / U_max (B.22) are taken over one x-y plane, which lies in the last slab: no reduction between slabs.
 * CLIP_ESTATE before clip_init, CLIP_EINVAL for a missing or misaligned buffer; clip_halo_bytes returns 0 for h == NULL. */
size_t clip_halo_bytes(const clip_t* h);
int clip_halo_pack(clip_t* h, void* d_lo, void* d_hi);
int clip_halo_unpack(clip_t* h, const void* d_recv_lo, const void* d_recv_hi, const void* d_sent_lo, const void* d_sent_hi);

/* Overlapped slab step: the exchange of a step's records runs on a second stream while the bulk of the step still computes.
 *   clip_halo_stream(h, s2)            s2 (cudaStream_t as void*, ideally of higher priority) becomes the handle's halo stream
 *                                      (NULL: none); the library creates three events for the ordering below.
 *   clip_step_halo_begin(h, d_lo, d_hi)  ONE time step.  k_fused path: the first and the last z chunk (the planes next to the HALO
 *                                      faces) run on the halo stream, followed there by clip_halo_pack into d_lo / d_hi; the other
 *                                      chunks and k_fix run on the handle's stream at the same time.  Other kernel paths: the step
 *                                      on the handle's stream, then the pack on the halo stream.  On return the records are being
 *                                      produced ON THE HALO STREAM: the caller enqueues its transfer there.
 *   clip_step_halo_end(h, recv_lo, recv_hi, sent_lo, sent_hi)   makes the handle's stream wait for the halo stream (the transfer)
 *                                      and runs clip_halo_unpack there.
 * CLIP_ESTATE without a halo stream or when begin / end do not alternate. */
int clip_halo_stream(clip_t* h, void* cuda_stream);
int clip_step_halo_begin(clip_t* h, void* d_lo, void* d_hi);
int clip_step_halo_end(clip_t* h, const void* d_recv_lo, const void* d_recv_hi, const void* d_sent_lo, const void* d_sent_hi);

/* Free the handle (not the workspace). */
int clip_destroy(clip_t* h);

/* Last error text of the handle, or of the last failed clip_create / clip_workspace_bytes when h == NULL.
 * The string is owned by the library and valid until the next call on that handle. */
const char* clip_last_error(const clip_t* h);

/* Number of kernel launches the handle has enqueued so far (instrumentation for bench.py's gpu_launches). */
long long clip_launch_count(const clip_t* h);

/* Number of time steps the handle has run by replaying its CUDA graph (instrumentation; see clip_step). */
long long clip_graph_steps(const clip_t* h);

/* Instrumentation for bench.py's roofline: like clip_step(h, n), but every kernel launch is bracketed by CUDA
 * events on the handle's stream; after synchronising the stream (this call is host-synchronous) the elapsed
 * milliseconds and launch counts are ADDED per kernel kind into ms[kind] / count[kind], kind < clip_kernel_kinds().
 * clip_kernel_name(kind) is the kernel's name (library-owned string), NULL if kind is out of range. */
int clip_step_profiled(clip_t* h, int n, double* ms, long long* count);
int clip_kernel_kinds(void);
const char* clip_kernel_name(int kind);

/* ---- no-allocation entry point --------------------------------------------------------------------------------------------------
 * For callers that may not allocate device memory at all (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc) and therefore cannot provide a workspace: lambda of the convective outlet for the step t -> t+1 (App. B.5: B.22 with
 * the three schemes U_local / U_ave / U_max; lambda = U dt / dx of B.25; U from the stored velocity of
 * the previous time step, i.e. outlet_u_time = 0; outlet_clamp as in clip_params, reading R12) -- what
 * k_outlet_lam + k_outlet_reduce compute inside clip_step for a lattice with an OUTLET on +z, with the same reduction order.
 *   d_u       device, [3][nz][ny][nx] words of `precision` (the layout clip_get writes): u(t); only u_z of layer nz-2 is read
 *   d_lambda  device, [ny][nx] words: receives lambda (uniform over the plane for outlet_u_mode 1 and 2)
 * Both aligned to the word size and owned by the caller; the two kernels are enqueued on `cuda_stream` (cudaStream_t as void*, NULL =
 * the default stream) of the CURRENT device, no host synchronisation.
 * The per-column scratch of the reduction lives in a static device array inside the library (2 MiB per GPU that loads the library,
 * held until exit), hence the limit nx * ny <= CLIP_STATIC_MAX_PLANE_NODES; larger planes are refused with CLIP_EINVAL.  Every call on
 * a device shares that array: calls that may overlap on the GPU (different streams without an ordering between them) race and must
 * be serialised by the caller; calls on one stream, or on different devices, are safe.  The array needs no clearing: each call
 * writes every entry it later reads.  Calls no cudaMalloc / cudaFree or other allocating routine.
 * Returns CLIP_OK, CLIP_EINVAL (sizes, modes, pointers) or CLIP_ECUDA; text via clip_static_last_error() (per host thread,
 * library-owned, valid until that thread's next call of clip_outlet_lambda_static). */
#define CLIP_STATIC_MAX_PLANE_NODES 262144
int clip_outlet_lambda_static(const void* d_u, int nx, int ny, int nz, int precision, int outlet_u_mode, int outlet_clamp,
                              void* d_lambda, void* cuda_stream);
const char* clip_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* CLIP_H_ */
