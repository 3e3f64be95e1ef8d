/*
 * dr.h -- C ABI of libdr: pseudo-transient (PT) solver for quasi-static linear elasticity on a 3-D voxel
 * image and the six-load-case driver that returns the effective 6x6 stiffness tensor (arXiv 2410.20441).
 *
 * Citations: P:NNN = PAPER.md line NNN of the paper text; "Reading Rn" = DESIGN.md section 3.
 *
 * Problem (sec. 2): div sigma = 0, sigma = C(x):eps(u) on a cuboid of nx*ny*nz cubic voxels of
 * size h with bulk modulus K and shear modulus G per voxel; apply a uniform strain through displacement
 * ("velocity", physical step Delta t = 1) boundary conditions (sec. 3.4, App. A);
 * <sigma> = C* <eps> (Eq. 7-9) gives one column of C* per load case.
 * Method (sec. 3.1): accelerated pseudo-transient iteration, Eq. 10-21, on a staggered grid
 * (sec. 3.3): normal stresses and moduli at cell centres, velocities on faces, shear stresses on edges.
 *
 * Conventions
 *  - All arrays are fp64, x fastest: index = i + nx*(j + ny*k) for the nx*ny*nz cell fields.
 *  - Voigt order xx,yy,zz,yz,xz,xy ("C55 (xz)" P:365); engineering shear strain gamma = 2 eps.
 *  - Load cases 0..5 apply the displacement gradient D with one non-zero entry eps0:
 *      0: Dxx  1: Dyy  2: Dzz  (normal compression tests, App. A.1)
 *      3: u_y = eps0 z   4: u_x = eps0 z   5: u_x = eps0 y   (simple shear tests, App. A.2)
 *    Load case 6 (dr_solve / dr_step only) is the 7th, triaxial test of App. A.3: Dxx = Dyy = Dzz = eps0 (dr_offdiag_direct).
 *  - Units of C* are the units of K and G.
 *  - The library allocates NO device memory: the caller passes one workspace of dr_workspace_bytes() bytes
 *    (e.g. a torch tensor) that is borrowed until dr_destroy.  K and G are borrowed during dr_create only.
 *  - A handle belongs to the CUDA device that was current at dr_create (the device of the workspace and the stream);
 *    every call switches to it and restores the caller's device on return.
 *  - Every launch goes to the cuda_stream given at dr_create (a cudaStream_t cast to void*, NULL = default
 *    stream).  Calls that return host values synchronise that stream.
 *  - Errors are return codes, never exceptions or aborts.  dr_last_error() gives a message for the last
 *    non-OK status of that handle.  DR_MAXITER is a soft status: fields, averages and the C column are
 *    valid and stored.
 *  - There is no CPU fallback: without a CUDA device every compute call returns DR_ERR_CUDA.
 */
#ifndef DR_H
#define DR_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dr_handle dr_handle;            /* opaque, owned by the library */

typedef enum {
    DR_OK = 0,
    DR_ERR_ARG = 1,         /* invalid argument (sizes, h<=0, eps0==0, tol<=0, negative/NaN moduli, ...)   */
    DR_ERR_WORKSPACE = 2,   /* workspace NULL, misaligned (needs 256 B) or smaller than dr_workspace_bytes */
    DR_ERR_CUDA = 3,        /* a CUDA runtime call failed (message in dr_last_error)                      */
    DR_ERR_DIVERGED = 4,    /* residual became NaN/Inf                                                     */
    DR_ERR_STATE = 5,       /* call order (e.g. dr_effective_C before six columns exist)                   */
    DR_MAXITER = 6          /* soft: maxiter reached before res <= tol                                     */
} dr_status;

/* dr_set_param ids.  Defaults in brackets. */
typedef enum {
    DR_CFL = 0,        /* C~ of Eq. 14 P:98 [0.55]; the 3-D stability limit is 1/sqrt(3) (Reading R10)        */
    DR_ST_FACTOR = 1,  /* St = 2 pi sqrt(3) * factor, Eq. 16, 21 P:107-130 [1.0]                               */
    DR_NCHECK = 2,     /* residual is evaluated every ncheck iterations [50]                                  */
    DR_GAVG = 3,       /* shear modulus on edges: 0 harmonic mean of the 4 cells [default], 1 arithmetic (R4) */
    DR_VOID_REL = 4,   /* r>0: cells with K+4G/3 <= r*max(K+4G/3) become exact void K=G=0 [0 = off] (R9)      */
    DR_BC_MODE = 5,    /* 0 paper's mixed BCs [default]; 1 full kinematic uniform BC on all faces (R5)        */
    DR_KERNEL = 6,     /* 0 fused z-march kernel with TMA staging; 1 split stress/velocity kernels
                          (baseline); 2 fused z-march kernel with register-prefetched LDG loads;
                          3 [default] temporal blocking: TWO PT iterations per sweep (the state is read and written once per two
                          iterations) on stencil-coded images -- images with <= 256 distinct (K,G) pairs, edge moduli
                          and node stiffnesses, i.e. segmented rock images; odd leftovers and a check iteration that
                          would be the first of a pair run one iteration of the same coded kernel; images that cannot be
                          coded run kernel 0 (dr_active_kernel tells), and so does DR_FORM 1;
                          4 one iteration per sweep with the coded kernel (A/B reference of 3)                          */
    DR_ZCHUNK = 7,     /* z layers per CTA of the fused kernels; 0 = automatic [default] (tuning knob)            */
    DR_PALETTE = 9,    /* 1 [default]: images with <= 256 distinct (K,G) pairs run the fused kernel on a uint8 phase id
                          per cell and a 256-entry table instead of the two fp64 modulus fields (same values, 14 B less
                          HBM traffic per voxel-iteration); 0: always the fp64 modulus fields                        */
    DR_STAG_TOL = 10,  /* second stopping rule of dr_solve (Reading R9b; the paper gives no rule beyond P:78): at every residual
                          check with res > tol the volume averages <sigma> (Eq. 7) are formed; two consecutive checks that
                          moved them by <= stag_tol (relative, max-norm over the 6 components) end the solve with DR_OK and
                          dr_stop_reason() = DR_STOP_STAGNATION [1e-10; 0 = off].  The movement is taken over at least 50
                          iterations: checks closer than that to the last comparison are skipped by this rule, so the
                          stop does not depend on DR_NCHECK when it is small (for DR_NCHECK >= 50 every check compares).
                          It ends solves whose max-norm plateaus in near-void pores (contrast 1e-6) while C* is converged;
                          DR_VOID_REL stays opt-in because it changes the moduli.  A solve ended this way returns DR_OK with
                          a residual ABOVE tol: read dr_stop_reason / dr_info_lc to tell the two apart                     */
    DR_FORM = 8        /* 0 stress-relaxation form of the paper, Eq. 11-13 [default]; 1 displacement form: state u, w,
                          w <- (1-theta) w + C~^2 h^2 F(u)/H_node, u <- u + w, stresses formed on the fly (same fixed
                          point, 112 instead of 160 B per voxel-iteration; DR_KERNEL 0 or 1).  Setting DR_FORM also resets
                          DR_CFL to the form's default (0.55 / 0.50: the explicit damping has less stability margin) */
} dr_param;

/* which rule ended the last dr_solve on a handle (dr_stop_reason) */
typedef enum {
    DR_STOP_NONE = 0,        /* no solve yet, or the solve diverged                                   */
    DR_STOP_RESIDUAL = 1,    /* res <= tol                                                       */
    DR_STOP_STAGNATION = 2,  /* <sigma> stopped moving between residual checks (DR_STAG_TOL)            */
    DR_STOP_MAXITER = 3      /* neither: maxiter reached (status DR_MAXITER)                            */
} dr_stop;

/* Bytes of device workspace dr_create needs for an nx*ny*nz grid (0 if the sizes are invalid). */
size_t dr_workspace_bytes(int nx, int ny, int nz);

/* Bytes of device workspace for a handle that can also run dr_solve_all: six state sets instead of one (0 if the sizes are
 * invalid).  191^3: 7.7 GB, 479^3: 111.5 GB, 703^3 does not fit one B200 -- the batch is meant for small and medium grids. */
size_t dr_workspace_bytes_six(int nx, int ny, int nz);

/* Create a solver.  nx,ny,nz >= 2; h > 0.
 * K, G: DEVICE pointers, nx*ny*nz doubles each, x fastest, >= 0 and finite (K = G = 0 is void, G = 0 with K > 0
 * is a fluid; both allowed).  They are read (copied into the workspace with a replicate halo) and not kept.
 * workspace: DEVICE pointer, 256-byte aligned, workspace_bytes >= dr_workspace_bytes(nx,ny,nz), borrowed until
 * dr_destroy; its previous content is overwritten.  cuda_stream: cudaStream_t or NULL.
 * Sets up the constants of Eq. 14-21.  On error *out = NULL. */
dr_status dr_create(int nx, int ny, int nz, double h,
                    const double* K, const double* G,
                    void* workspace, size_t workspace_bytes,
                    void* cuda_stream, dr_handle** out);

/* The same for a SEGMENTED image, the usual product of CT segmentation (the marble image is a phase map):
 * phase: DEVICE pointer, nx*ny*nz bytes, x fastest, phase id of every cell (0 .. nphase-1; an id >= nphase is DR_ERR_ARG);
 * 1 <= nphase <= 256; K_table, G_table: HOST pointers, nphase doubles each (same value rules as dr_create).  The handle is
 * identical, bit for bit, to the one dr_create builds from the expanded arrays K = K_table[phase], G = G_table[phase]; the
 * caller moves 1 byte per cell instead of 16. */
dr_status dr_create_segmented(int nx, int ny, int nz, double h,
                              const unsigned char* phase, int nphase, const double* K_table, const double* G_table,
                              void* workspace, size_t workspace_bytes,
                              void* cuda_stream, dr_handle** out);

/* Set a parameter (before dr_solve / dr_step).  Changing a parameter that shapes the iterate (DR_CFL, DR_ST_FACTOR,
 * DR_GAVG, DR_VOID_REL, DR_BC_MODE, DR_KERNEL, DR_FORM) discards the current fields: dr_iterate / dr_get_field return
 * DR_ERR_STATE until the next dr_step / dr_solve. */
dr_status dr_set_param(dr_handle* h, int id, double value);

/* One load case: initial fields and boundary values (App. A), then PT iterations (Eq. 11-13) until the
 * residual max-norm  res = max_nodes |div sigma| h / (H_node |eps0|)  <= tol, tested every ncheck iterations
 * ("once the dynamic fields attenuate to a certain precision"), or until <sigma> has stopped moving
 * (DR_STAG_TOL), at most maxiter iterations; then the
 * volume averages (Eq. 7) and column load_case of C* (Eq. 9, 22).  eps0 != 0, tol > 0, maxiter >= 1. */
dr_status dr_solve(dr_handle* h, int load_case, double eps0, double tol, int maxiter);

/* The six load cases of the image advanced together on ONE handle (one direct test per stiffness column; the
 * tests share K and G): every launch of the two-iteration kernel carries all load cases that have not met a stopping rule
 * yet, so a small grid fills the GPU and needs a sixth of the launches.  Needs a workspace of dr_workspace_bytes_six() bytes
 * at dr_create (else DR_ERR_WORKSPACE).  Same iterates, checks, stopping rules and C* as six dr_solve calls (on images that
 * cannot be stencil-coded, or with DR_KERNEL != 3 / DR_FORM 1, it simply runs those six calls).  status_out: HOST, 6 ints
 * (dr_status per load case) or NULL.  Returns the worst status; afterwards dr_effective_C and dr_info_lc are valid
 * (dr_get_field is not: call dr_step / dr_solve for fields). */
dr_status dr_solve_all(dr_handle* h, double eps0, double tol, int maxiter, int status_out[6]);

/* Iterations done, last residual and dr_stop value of load case lc (0..5) in the last dr_solve_all.  Pointers may be NULL. */
dr_status dr_info_lc(dr_handle* h, int load_case, int* iters, double* residual, int* stop);

/* The six load cases at once on six solvers (h[lc] solves load case lc; six distinct handles, each with its own
 * workspace and, to overlap on the device, its own stream).  One host thread enqueues every unfinished load case up
 * to its next residual check before it waits for any of them, so small grids that cannot fill the GPU alone run
 * concurrently (one direct test per stiffness column).  Same iterates and stopping rule as six dr_solve
 * calls.  status_out: HOST, 6 ints (dr_status per load case) or NULL.  Returns the worst status. */
dr_status dr_solve_six(dr_handle* const h[6], double eps0, double tol, int maxiter, int status_out[6]);

/* C* (HOST, row-major out[6*m + n]) with column n taken from h[n], after dr_solve_six. */
dr_status dr_effective_C_six(dr_handle* const h[6], double out[36]);

/* Same with a fixed iteration count and no convergence test (parity tests): initial fields, niter >= 0
 * iterations, the residual of the last iteration, the volume averages and the (unconverged) column. */
dr_status dr_step(dr_handle* h, int load_case, double eps0, int niter);

/* Continue niter PT iterations from the current fields without residual or averages (throughput timing).
 * Needs a previous dr_step/dr_solve with the same load case and eps0.  Does not synchronise the stream. */
dr_status dr_iterate(dr_handle* h, int load_case, double eps0, int niter);

/* Effective stiffness, HOST pointer, row-major out[6*m + n] = C*_mn (Voigt).  DR_ERR_STATE until all six
 * load cases have been solved.  Not symmetrised. */
dr_status dr_effective_C(dr_handle* h, double out[36]);

/* The paper's 7th direct test (App. A.3).  load_case 6 of dr_solve / dr_step prescribes the normal displacement
 * of all three face pairs at once (Dxx = Dyy = Dzz = eps0; tangential components free as in the normal tests).  After load
 * cases 0, 1, 2 and 6 have been solved on this handle, Eq. 24-29 give the off-diagonal normal components from
 * sigma_bar_k = <sigma_kk> - C_kk eps_k and eps_bar_k = eps0:  out = (C12, C13, C23), HOST pointer.  The problem is linear,
 * so these equal the symmetrised off-diagonals of dr_effective_C to solver tolerance (a consistency diagnostic; the six
 * columns already hold C12, C13, C23).  DR_ERR_STATE until the four load cases exist.  Load case 6 is not part of
 * dr_effective_C, dr_solve_all or dr_solve_six. */
dr_status dr_offdiag_direct(dr_handle* h, double out[3]);

/* Volume-averaged stresses of the last solve/step, HOST pointer, Voigt order (Eq. 7). */
dr_status dr_avg_stress(dr_handle* h, double out[6]);

/* Volume-averaged stresses (Eq. 7, Reading R7: cell sum of the normal stresses, trapezoid weights on the edge shears)
 * of six DENSE device fields, WITHOUT a handle, a workspace or any allocation.
 *
 * Why it exists.  Every other compute call works in a workspace the caller allocated.  Some callers have no way to get
 * one: a progress or post-processing hook running beside a long solve, where a cudaMalloc / cudaFree would serialise
 * against all work on the device and stall the solver's streams each time; or a plug-in inside a host program whose
 * allocator already holds whatever device memory a large image leaves free, so that an allocation of the plug-in's own
 * fails.  For them the reduction scratch is a fixed 6 MiB array compiled into libdr.so itself.  Every GPU on which the
 * library's device code gets loaded carries these 6 MiB until the process exits, whether or not this call is ever used.
 *
 * Arguments.  stress: HOST array of six DEVICE pointers in Voigt order, each a dense x-fastest array as dr_get_field
 * writes it: sxx, syy, szz (nx,ny,nz), tyz (nx,ny+1,nz+1), txz (nx+1,ny,nz+1), txy (nx+1,ny+1,nz); read only, borrowed until
 * the work enqueued by this call has run.  out6: DEVICE, 6 doubles, written by the last kernel of the call.  cuda_stream:
 * cudaStream_t or NULL; both kernels go there and the call does NOT synchronise -- read out6 in stream order.  All pointers
 * and the stream belong to the CURRENT device (there is no handle to remember one).  errbuf: HOST, errbuf_len bytes, or
 * NULL; receives a message whenever the return value is not DR_OK (emptied on success).
 *
 * Limit.  (ny+1)*(nz+1) <= DR_STATIC_MAX_ROWS (the scratch holds six partial sums per eight x-rows); nx, ny, nz in 2..8192.
 * That covers every cube up to 1023^3 (all five benchmark images).  A larger grid is refused with DR_ERR_ARG and a message
 * that names the limit; nothing is launched.  Use a handle and dr_avg_stress there.
 *
 * First call.  The first call on each device looks up that device's address of the built-in array
 * (cudaGetSymbolAddress, checked; DR_ERR_CUDA if it fails) and keeps it for the process.  Make that first call during
 * set-up, before any stream capture is begun.  Later calls only launch two kernels.  No cudaMalloc, cudaFree, host
 * allocation or allocating library routine is called on any path.
 *
 * Sharing.  There is ONE array per device and every call uses it.  It is not cleared: a call overwrites the part it will
 * read, so nothing has to start at zero and whatever an earlier call left is never looked at.  Two calls whose kernels can
 * overlap on the GPU (different streams, or different host threads on different streams) write the same partial sums and
 * both results are then garbage -- keep all calls on one stream, or order them with events.
 *
 * Result.  Same weights and the same quantity as dr_avg_stress after dr_step / dr_solve on the fields of that handle; the sum is
 * grouped differently (by eight rows instead of by a fixed number of blocks), so the two agree to rounding, not bit for
 * bit.  Run-to-run deterministic.  Without a CUDA device: DR_ERR_CUDA. */
#define DR_STATIC_MAX_ROWS 1048576
dr_status dr_avg_stress_static(int nx, int ny, int nz, const double* const stress[6], double* out6,
                               void* cuda_stream, char* errbuf, size_t errbuf_len);

/* Iterations done, last residual, and milliseconds (CUDA events on the stream, whole call) of the last
 * dr_solve/dr_step.  Any pointer may be NULL. */
dr_status dr_info(dr_handle* h, int* iters, double* residual, double* ms);

/* Copy one field to a dense DEVICE array of its logical shape (x fastest, no pitch):
 * field 0 vx (nx+1,ny,nz)   1 vy (nx,ny+1,nz)   2 vz (nx,ny,nz+1)   3 sxx  4 syy  5 szz (nx,ny,nz)
 *       6 tyz (nx,ny+1,nz+1)   7 txz (nx+1,ny,nz+1)   8 txy (nx+1,ny+1,nz);   sigma_aa = -p + tau_aa (Eq. 10).
 * n must equal the number of elements of that shape. */
dr_status dr_get_field(dr_handle* h, int field, double* dst_device, size_t n);

/* Whole 6x6 tensor from HOST arrays through the public API with host<->device copies inside: allocates
 * nothing on the device itself -- K_host/G_host (nx*ny*nz doubles, pinned or pageable) are staged through
 * stage_device (DEVICE, >= 2*nx*ny*nz doubles, caller-owned), then dr_create + the six load cases + dr_effective_C
 * run in `workspace` (dr_solve_all if it has dr_workspace_bytes_six() bytes, else six dr_solve calls).  C_out: HOST, 36 doubles.  iters_out: HOST, 6 ints or NULL.  Returns the worst status. */
dr_status dr_solve_image_host(int nx, int ny, int nz, double h,
                              const double* K_host, const double* G_host,
                              double* stage_device, void* workspace, size_t workspace_bytes, void* cuda_stream,
                              double eps0, double tol, int maxiter, int ncheck,
                              double C_out[36], int iters_out[6]);

/* dr_solve_image_host for a segmented image: phase_host (HOST, nx*ny*nz bytes) is staged through stage_device (DEVICE,
 * >= nx*ny*nz bytes, caller-owned), then dr_create_segmented and the six load cases as above. */
dr_status dr_solve_image_host_segmented(int nx, int ny, int nz, double h,
                                        const unsigned char* phase_host, int nphase, const double* K_table, const double* G_table,
                                        unsigned char* stage_device, void* workspace, size_t workspace_bytes, void* cuda_stream,
                                        double eps0, double tol, int maxiter, int ncheck,
                                        double C_out[36], int iters_out[6]);

/* Compliance (property) contribution tensor of the inclusions, Eq. 23: S* = S1 + phi H, i.e.
 * H = ((C*)^-1 - (C1)^-1) / phi.  Pure host post-processing of two effective tensors (the image and the matrix-only
 * run, BASELINE config 2): all pointers HOST, 6x6 row-major, Voigt with engineering shear; 0 < phi <= 1 is the
 * inclusion volume fraction.  DR_ERR_ARG if an argument is NULL/out of range or a matrix is singular. */
dr_status dr_contribution_tensor(const double C_eff[36], const double C_matrix[36], double phi, double H_out[36]);

/* 1 if dr_solve / dr_step on this handle run the phase-id (palette) variant of the fused kernel (the image has at
 * most 256 distinct (K,G) pairs, DR_PALETTE = 1, DR_KERNEL = 0), else 0. */
int dr_uses_palette(dr_handle* h);

/* Kernel the iterations on this handle run with the current parameters and image (see DR_KERNEL; valid after
 * dr_step / dr_solve).  -1 for a NULL handle. */
int dr_active_kernel(dr_handle* h);

/* dr_stop value of the last dr_solve / dr_solve_six on this handle: which stopping rule fired. */
int dr_stop_reason(dr_handle* h);

/* Number of kernel launches this handle has issued so far (for bench.py's gpu_launches). */
long long dr_launch_count(dr_handle* h);

const char* dr_last_error(dr_handle* h);

void dr_destroy(dr_handle* h);

#ifdef __cplusplus
}
#endif
#endif /* DR_H */
