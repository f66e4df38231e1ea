/* lb.h -- C ABI of the B200-native two-component Shan-Chen D3Q19 lattice-Boltzmann library.
 *
 * One library, one GPU, one opaque context per simulation box.  Every step of the hot
 * path (moments, Shan-Chen force, BGK collision with forcing, halfway bounce-back,
 * periodic streaming, diagnostics) runs in hand-written sm_100a CUDA kernels behind
 * these calls.  There is no CPU fallback: with no CUDA device every call that touches
 * the device fails with LB_ECUDA.
 *
 * Citations: PAPER.md = /root/reference/PAPER.md (LBcuda, arXiv 2112.08264);
 * S1..S14 = the readings of SURVEY.md 8(c), repeated in DESIGN.md "Readings".
 *
 * CONVENTIONS
 *   Box        nx*ny*nz nodes, periodic on all three axes (section 5).
 *   Node index n = x + nx*(y + ny*z); every array argument is dense, x fastest, no
 *              padding.  N = nx*ny*nz.
 *   Components k = 0 "red", k = 1 "blue".
 *   Directions i = 0..18, D3Q19, numbered (reading S1):
 *              0:(0,0,0)  1:(+x) 2:(-x) 3:(+y) 4:(-y) 5:(+z) 6:(-z)
 *              7:(+x+y) 8:(-x-y) 9:(+x-y) 10:(-x+y)
 *              11:(+x+z) 12:(-x-z) 13:(+x-z) 14:(-x+z)
 *              15:(+y+z) 16:(-y-z) 17:(+y-z) 18:(-y+z);  opp(i) = i+1 (i odd), i-1 (i even >= 2).
 *   Pointers   every pointer argument is a caller-owned HOST array (pageable or pinned).
 *              The library copies; it never keeps a caller pointer after the call returns.
 *              All device state is owned by the context; its layout is private.
 *   Values     the ABI speaks double for both LB_F64 and LB_F32 contexts; an LB_F32 context
 *              rounds to float on the way in and widens on the way out.
 *   Errors     lb_create* return NULL on failure; all other calls return LB_OK or a negative
 *              code; lb_last_error() holds a message and lb_last_error_code() the code of the
 *              last failure on the calling thread.  No exception crosses the boundary.
 *   Device     a context lives on the CUDA device that is current when it is created; every
 *              later call switches to that device for its own duration.
 *   Ordering   lb_step only enqueues work on the context's stream and may return before the
 *              GPU finishes; every getter synchronises that stream.
 *   Threads    one context may be used from one thread at a time.
 */
#ifndef LB_B200_H
#define LB_B200_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lb_ctx lb_ctx;          /* opaque; owned by the library */

enum { LB_OK = 0, LB_EINVAL = -1, LB_ENOMEM = -2, LB_ECUDA = -3, LB_ESTATE = -4 };
enum { LB_F64 = 0, LB_F32 = 1 };
enum { LB_KERNEL_AUTO = 0, LB_KERNEL_TWOPASS = 1, LB_KERNEL_ONEPASS = 2, LB_KERNEL_TMA = 3, LB_KERNEL_HALO = 4, LB_KERNEL_NODE = 5 };
enum { LB_OPT_ZC = 1, LB_OPT_DIAG = 2, LB_OPT_BALANCE = 3 };
enum { LB_MODEL_SHAN_CHEN = 0, LB_MODEL_COLOUR_GRADIENT = 1 };   /* options of lb_set_option */

/* Create a context for an nx*ny*nz periodic box holding two fluids with BGK
 * relaxation times tau_r, tau_b (Eq. 1; omega_k = 1/tau_k) coupled by the
 * Shan-Chen constant G (reading S2: F^k(x) = -G psi^k(x) sum_{i=1..18} w_i psi^kbar(x+c_i) c_i,
 * psi = rho (S3), w_i the lattice weights of PAPER.md:393-398; G > 0 repels).
 * fp64 populations, the library's own stream.
 * NULL (LB_EINVAL) if a dimension is < 1, ny or nz > 65535, N >= 2^31, tau <= 0.5 or not finite (Eq. 2, PAPER.md:84-86,
 * needs 0 < omega < 2), or G is not finite; NULL (LB_ENOMEM / LB_ECUDA) if device memory or
 * the device is not available; lb_last_error_code() tells which.  Device memory: 2 population
 * buffers of 38*N values; the carried density, 2 x 2 arrays of N values plus tile-edge arrays
 * and, for LB_KERNEL_HALO, 2 x 20/32 N values of x-halo copies (about 70 bytes per node in fp64,
 * 35 in fp32, when nx % 32 == 0 and ny % 8 == 0; 32 / 16 otherwise); 4 bytes per node of link
 * words; a staging buffer of 40 bytes x min(N, 2^22). */
lb_ctx* lb_create(int nx, int ny, int nz, double tau_r, double tau_b, double G);

/* Same, with the population type (LB_F64 / LB_F32: "fp32 populations and fields", all
 * arithmetic in that type) and, if cuda_stream != NULL, a caller-owned cudaStream_t on
 * which all the context's work is enqueued (e.g. a torch stream); the caller keeps that
 * stream alive until lb_destroy. */
lb_ctx* lb_create_ex(int nx, int ny, int nz, double tau_r, double tau_b, double G,
                     int dtype, void* cuda_stream);

/* Release the context and all its device memory.  lb_destroy(NULL) is a no-op. */
void lb_destroy(lb_ctx* ctx);

/* Initialise both fluids at local equilibrium (Eq. 10, c_s^2 = 1/3):
 * f_i^k(x) = f_i^eq(rho^k(x), u(x)).  rho_r, rho_b: N doubles each (required).
 * ux, uy, uz: N doubles each, or all three NULL for u = 0.  Solid nodes get exactly 0 (S8).
 * LB_EINVAL on NULL rho pointers or a partial velocity triple. */
int lb_set_fields(lb_ctx* ctx, const double* rho_r, const double* rho_b,
                  const double* ux, const double* uy, const double* uz);

/* Static solid nodes (nodes inside particles, "no computation is
 * performed"): N bytes, nonzero = solid.  May be called before or after lb_set_fields; either
 * way solid-node populations are exactly 0 afterwards (S8).  Fluid->solid links get halfway
 * bounce-back with the wall at rest (Eq. 23-24 with u_b = 0); a solid
 * neighbour contributes psi = 0 to the force sum (S7). */
int lb_set_solid_mask(lb_ctx* ctx, const unsigned char* mask);

/* Restart / arbitrary state: 38*N doubles, [k][i][z][y][x].  Solid nodes are zeroed. */
int lb_set_populations(lb_ctx* ctx, const double* f);

/* Advance nsteps time steps.  One step, for every fluid node x (order of PAPER.md:128-138:
 * collide -> bounce-back -> stream):
 *   rho^k = sum_i f_i^k, j^k = sum_i f_i^k c_i                          (Eq. 6-7)
 *   u'    = sum_k omega_k j^k / sum_k omega_k rho^k                     (S4; Eq. 7 when tau_r = tau_b)
 *   du^k  = -G sum_{i=1..18} w_i rho^kbar((x+c_i) mod box) c_i          (S2, S3, S6, S7)
 *   f*_i  = (1-omega_k) f_i + omega_k feq_i(rho^k,u') + feq_i(rho^k,u'+du^k) - feq_i(rho^k,u')   (Eq. 1 + S5)
 *   x+c_i solid: f_opp(i)^k(x,t+1) = f*_i  else  f_i^k((x+c_i) mod box, t+1) = f*_i              (Eq. 23-24; Eq. 5)
 * Solid nodes keep 0.  LB_EINVAL if nsteps < 0; LB_ESTATE before lb_set_fields /
 * lb_set_populations; LB_ECUDA on a launch failure.  Asynchronous. */
int lb_step(lb_ctx* ctx, int nsteps);

/* Copy out all populations: 38*N doubles, [k][i][z][y][x].  Synchronises. */
int lb_get_populations(lb_ctx* ctx, double* f);

/* rho^k (Eq. 6) and the barycentric velocity u = sum_k j^k / sum_k rho^k (Eq. 7) of the current
 * state; N doubles each; any pointer may be NULL to skip that field.  Solid nodes and nodes
 * with zero total density report 0.  Synchronises. */
int lb_get_moments(lb_ctx* ctx, double* rho_r, double* rho_b, double* ux, double* uy, double* uz);

/* Bounce-back link set: N 32-bit words; bit i of links[n] is set iff node n is fluid and
 * (n + c_i) mod box is solid.  Integer work: exactly one right answer.  Synchronises. */
int lb_get_link_mask(lb_ctx* ctx, unsigned int* links);

/* Per-component mass M^k = sum_x rho^k and total momentum P = sum_x sum_k j^k over fluid nodes
 * of the current state (warp-shuffle + fixed-order block reduction: deterministic).
 * Accumulated in double for both dtypes.  Synchronises. */
int lb_get_diagnostics(lb_ctx* ctx, double mass[2], double momentum[3]);

/* lb_get_diagnostics for callers that cannot allocate or synchronise (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same two kernels (per-block partial sums of the moments of Eq. 6-7, then a
 * fixed-order final pass: deterministic), but the partials live in a static __device__ array of the library instead of
 * allocated memory, and the five sums {M^r, M^b, P_x, P_y, P_z} go to out_dev, DEVICE memory for 5 doubles owned by the
 * caller.  Calls no cudaMalloc, cudaFree, memcpy or synchronisation: two launches on the context's stream, the result is
 * there once the stream reaches that point.  Limit: boxes of at most 2^28 nodes (16384 partials of 16384 nodes each, 640 KB
 * of device memory that every GPU which loads the library holds until the process exits); a larger box is LB_EINVAL with
 * a message saying so.  Every call on a device shares that array and finds the last call's contents in it (nothing has to
 * start at zero: each block overwrites its own partial): calls whose kernels overlap on the GPU (different streams of one
 * device) race; calls on one stream, or ordered by events, do not.  LB_ESTATE before lb_set_fields / lb_set_populations;
 * LB_ECUDA if the array's device address could not be obtained when the context was created. */
int lb_diagnostics_noalloc(lb_ctx* ctx, double* out_dev);

/* Choose the time-step kernel: LB_KERNEL_TWOPASS = density pass + fused collide/stream pass
 * (reads the populations twice per step); LB_KERNEL_ONEPASS = single fused pass that
 * reads and writes every population once per step, populations pulled with per-thread loads;
 * LB_KERNEL_TMA = the same single pass with the populations staged in shared memory by the TMA
 * unit (the fastest; needs nx % 32 == 0 and ny % 8 == 0 like ONEPASS); LB_KERNEL_HALO = a second
 * TMA-staged single pass that reads aligned tiles only (the x neighbour's column comes from
 * x-halo copies) and sums the density of the tile's own nodes from the staged populations
 * instead of carrying it (less DRAM traffic, measured slower; no bounce-back: a box with solid
 * nodes runs LB_KERNEL_TMA instead); LB_KERNEL_NODE = the TMA-staged single pass with one thread
 * per node doing both components (LB_KERNEL_TMA: one thread per node and component): a third fewer
 * instructions for the same bytes, no bounce-back (a box with solid nodes runs
 * LB_KERNEL_TMA instead); LB_KERNEL_AUTO (default) = the TMA-staged pass when the box shape allows
 * it (ONEPASS if the driver cannot encode the tensor maps), else TWOPASS: boxes whose sides are not
 * multiples of the 32 x 8 tile run about 1.5 x slower.  Under AUTO the library picks the thread
 * mapping itself: LB_KERNEL_NODE for an fp64 box (either operator) without solid nodes (measured 2 %
 * faster with Shan-Chen, 13 % with the colour gradient), LB_KERNEL_TMA otherwise;
 * lb_get_kernel reports which.  LB_EINVAL if the box shape does not allow `kind`. */
int lb_set_kernel(lb_ctx* ctx, int kind);

/* The kernel lb_step will use (LB_KERNEL_TWOPASS, LB_KERNEL_ONEPASS, LB_KERNEL_TMA, LB_KERNEL_HALO or LB_KERNEL_NODE; never AUTO);
 * -1 for a NULL context. */
int lb_get_kernel(const lb_ctx* ctx);

/* Tuning and modes.  LB_OPT_ZC: planes per CTA of the one-pass kernels (each CTA marches over
 * value z planes and re-collides one more at either end); 0 = the library's heuristic (default),
 * which also cuts the last few tile columns into one chunk more so that the TMA-staged kernels' CTA count
 * is a multiple of the SM count (an explicit value keeps every chunk at exactly `value` planes).
 * LB_OPT_DIAG (0 / 1, default 0): per-step diagnostics fused into the step: with LB_KERNEL_TMA,
 * LB_KERNEL_NODE and LB_KERNEL_HALO on a box without solid nodes (Shan-Chen operator), every lb_step leaves the per-component mass and the
 * total momentum of the NEW state behind (warp-shuffle reductions, one partial per CTA, added in
 * a fixed order: deterministic), and lb_get_diagnostics then makes no pass over the populations;
 * the momentum is the sum of the post-collision moments (1 - omega_k) j^k + omega_k rho^k u' +
 * rho^k du^k, which streaming in a periodic box only permutes.  Otherwise (solid nodes, other
 * kernels, other operators) lb_get_diagnostics makes its own pass as before.
 * LB_OPT_BALANCE (0 / 1, default 1): with LB_OPT_ZC left at 0, cut the last tile columns of the TMA-staged
 * kernels into one z chunk more so that their CTA count is a multiple of the SM count (whole waves; measured
 * 1 - 2 % faster); 0 keeps every column at the same number of chunks.
 * LB_EINVAL for an unknown option or a value out of range.  lb_get_option returns the value in
 * effect (for LB_OPT_ZC: the planes per CTA the current kernel will use), -1 on error. */
int lb_set_option(lb_ctx* ctx, int option, long long value);
long long lb_get_option(const lb_ctx* ctx, int option);

/* Number of kernel launches this context has enqueued so far (for bench.py's gpu_launches). */
long long lb_launch_count(const lb_ctx* ctx);

/* Block until all work enqueued on the context's stream has finished. */
int lb_sync(lb_ctx* ctx);

/* Message for the last failure on the calling thread ("" if none). */
const char* lb_last_error(void);

/* Code of the last failure on the calling thread (LB_OK if none): tells LB_EINVAL, LB_ENOMEM
 * and LB_ECUDA apart after lb_create* returned NULL. */
int lb_last_error_code(void);

/* Library version string. */
const char* lb_version(void);

/* ---- later operators (the paper's own two-fluid model and its moving walls) -----------------------------------------
 * Colour gradient runs in its own variants of the TMA-staged kernels on boxes without solid nodes that take the 32 x 8
 * tile (kernel choice AUTO, TMA or NODE; AUTO picks NODE in fp64: one colour-blind collision per node instead of one per
 * component), everything else (solid nodes, moving walls, other box shapes) on the general two-pass path.
 *
 * Colour-gradient collision (Eq. 8-21): replaces the Shan-Chen force + BGK of lb_step by
 *   Theta = (rho^1 - rho^2) / (rho^1 + rho^2), grad Theta = (1 / c_s^2) sum_i w_i Theta(x + c_i) c_i,
 *   omega = 2 / (6 nu + 1) with 1 / nu = (rho^1 / rho) / nu_1 + (rho^2 / rho) / nu_2, nu_k = c_s^2 (tau_k - 1/2),
 *   BGK with that omega towards feq_i(rho^k, u) (Eq. 9-10, u by Eq. 7), the perturbation of Eq. 17 with A = (9/4) sigma omega
 *   (Eq. 19) and the B_i of PAPER.md:393-398, and the recolouring of Eq. 20-21 with strength beta in [0, 1];
 * readings C1-C6 of DESIGN.md section 3 for what the paper leaves open or prints garbled.  G is ignored.  Streaming,
 * bounce-back, fields, getters and diagnostics are unchanged.  lb_set_shan_chen switches back.  LB_EINVAL for a
 * non-finite sigma or beta outside [0, 1]. */
int lb_set_colour_gradient(lb_ctx* ctx, double sigma, double beta);
int lb_set_shan_chen(lb_ctx* ctx);

/* Solid spheres with prescribed velocities (Eq. 22-27): np spheres of one radius, centres[np][3]
 * real-valued, vel[np][3] and omega[np][3] their translational and angular velocities (NULL = 0).  Sets the solid mask
 * (a node is solid iff its minimum-image squared distance to a centre <= radius^2, reading S9) like lb_set_solid_mask;
 * the geometry stays where it is, only the walls move: a link i from fluid node r into sphere p returns
 *   f_opp(i)^k(r, t+1) = f*_i^k(r) - 2 rho^k(r) w_i (u_b . c_i) / c_s^2,  u_b = v_p + r_b x omega_p,  r_b = r + c_i / 2 - centre_p
 * (Eq. 22, Eq. 24), and hands F_i = c_i [f*_i + f_opp(i)(t+1)] (both components) to the sphere (Eq. 25-26), with torque
 * F_i x r_b (Eq. 27); readings M1-M4 of DESIGN.md section 3.  lb_get_sphere_forces returns F[np][3], T[np][3] of the LAST
 * step, accumulated in fp64 for both dtypes with atomic adds (fp64 accumulators; the order of the sum is
 * not fixed, as the paper notes for its own GPU code at PAPER.md:240).  np = 0 removes the spheres and all solids;
 * lb_set_solid_mask afterwards also makes every solid a wall at rest again.  Synchronises. */
int lb_set_spheres(lb_ctx* ctx, int np, const double* centres, double radius, const double* vel, const double* omega);
int lb_get_sphere_forces(lb_ctx* ctx, double* F, double* T);

/* ---- slab decomposition ("equal sub-domains ... border exchange"; Tables 4-5) ----------------
 * The box of one context can be a z slab of a larger periodic box with two ghost planes on either side: run lb_step on
 * the slab as it is (its own periodic wrap only ever feeds the outermost ghost planes, whose results are thrown away)
 * and, before every step, overwrite the ghost planes with the neighbour slabs' outermost interior planes.  These two
 * calls move whole z planes [z0, z0 + nplanes) of the device state to / from a caller-owned DEVICE buffer of
 * lb_plane_buffer_bytes(ctx, nplanes) bytes (library-private content: the 38 population planes and, when the current
 * kernel carries the density from step to step (TMA, ONEPASS), that density of the same planes, so that the one-pass
 * kernels keep running on slabs), on the context's stream, asynchronously: the caller ships the buffer to the
 * neighbour rank (NCCL / peer copy over NVLink) on the same stream or after lb_sync.  Both ends must be contexts of
 * the same box cross-section, type and kernel.  paper_2112_08264_b200/slab.py drives this.
 * LB_EINVAL if the range leaves the box, LB_ESTATE before any state was set; lb_plane_buffer_bytes: -1 on error. */
int lb_export_planes(lb_ctx* ctx, int z0, int nplanes, void* device_dst);
int lb_import_planes(lb_ctx* ctx, int z0, int nplanes, const void* device_src);
long long lb_plane_buffer_bytes(const lb_ctx* ctx, int nplanes);

/* ---- single-fluid calibration path (the paper's case 1, Table 1) --------------
 * One BGK fluid on the same D3Q19 lattice, periodic box, no force, no solids, fused collide +
 * stream: f_i(x + c_i, t + 1) = (1 - omega) f_i + omega feq_i(rho, u) (Eq. 1, PAPER.md:77-80;
 * Eq. 10), 19 * 2 values moved per node and step (304 B in fp64, 152 B in fp32:
 * the paper's B = 19 x 2 x 8 per fluid).  Same conventions as above (host
 * pointers, dense [z][y][x] arrays, doubles at the boundary, error codes, lb_last_error).
 * Any box shape with ny, nz <= 65535.  Populations: 19 * N doubles, [i][z][y][x]. */
typedef struct lbs_ctx lbs_ctx;
lbs_ctx* lbs_create(int nx, int ny, int nz, double tau, int dtype, void* cuda_stream);   /* NULL on failure */
void lbs_destroy(lbs_ctx* ctx);
int  lbs_set_fields(lbs_ctx* ctx, const double* rho, const double* ux, const double* uy, const double* uz);   /* u: all NULL = 0 */
int  lbs_set_populations(lbs_ctx* ctx, const double* f);
int  lbs_step(lbs_ctx* ctx, int nsteps);                       /* asynchronous; LB_ESTATE before a set call */
int  lbs_get_populations(lbs_ctx* ctx, double* f);             /* synchronises */
int  lbs_get_moments(lbs_ctx* ctx, double* rho, double* ux, double* uy, double* uz);   /* any pointer may be NULL */
int  lbs_sync(lbs_ctx* ctx);
long long lbs_launch_count(const lbs_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* LB_B200_H */
