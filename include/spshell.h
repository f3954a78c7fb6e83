/*
 * spshell.h -- C ABI of the B200-native hot path of Bruegmann's CFF pseudospectral matrix method
 * for tensor fields on a spherical shell (arXiv:1104.3408; citations are PAPER.md:<line>).
 *
 * The library computes, entirely in hand-written FP64 CUDA kernels for sm_100a,
 *   (a) the Cartesian gradient of all evolved fields from the Chebyshev (radial) and double-Fourier
 *       (theta, phi) differentiation matrices plus the coordinate Jacobian (eq. 6-19);
 *   (b) the spin-weighted spherical-harmonic "Yn" tensor filter as matrix multiplication
 *       (eq. 46-62);
 *   (c) the right-hand side of the first-order scalar wave system with characteristic boundaries
 *       (config 5 of BASELINE.json; readings W1-W3).
 * There is no CPU fallback and no other backend: every hot call needs a CUDA device.
 *
 * STATE LAYOUT (PAPER.md:118 with the single cover, reading Q4).  Every state-shaped
 * array is `double`, linear index
 *        p = k + Nr*(i + Ntheta*(j + Nphi*mu)),
 * k = radial node (fastest), i = latitude, j = longitude, mu = field (slowest).  Grid (eq. 2-4):
 * r_k = (r_out+r_in)/2 - (r_out-r_in)/2 cos(pi k/(Nr-1)), theta_i = pi(i+1/2)/Ntheta,
 * phi_j = 2 pi j/Nphi, with Nphi = 2 Ntheta (eq. 5).
 *
 * POINTERS.  Arguments named *_dev are DEVICE pointers owned by the caller (PyTorch allocations in
 * the Python binding); *_host are host pointers.  The library owns only the sp_shell and the
 * device-resident matrix tables it uploaded in sp_build_matrices.  Hot calls allocate nothing, are
 * asynchronous on the given stream (a cudaStream_t passed as void*, NULL = default stream), do not
 * synchronise, and are deterministic (no atomics): same inputs give bit-identical outputs.
 *
 * CONCURRENCY.  A shell owns one internal side stream and two events with which independent launches of one call
 * (cosine / sine products, real / complex theta products, tensor groups) are forked from and joined to the caller's
 * stream; this is legal under CUDA stream capture, so hot calls can be captured into CUDA graphs.  Calls on the same
 * shell may be issued on different streams (e.g. the gradient on one, the filter on another), but from ONE host thread
 * at a time: the shell's events are not protected against concurrent host threads.  Different shells are independent.
 *
 * ERRORS.  Every call returns an sp_status; nothing throws across the ABI.  Argument errors are detected before anything is launched
 * and leave the outputs untouched.  After any other non-OK status of a hot call (SP_ERR_CUDA: a launch failed mid-pipeline) the
 * contents of the output arrays and of the workspace are UNDEFINED (earlier stages may have written intermediates into them, e.g. the
 * gradient's d/dx slot); the shell's side stream is joined back into the caller's stream on every exit path, so a failed call
 * cannot leave a CUDA graph capture forked.  Several shells may live in one process, built in any order, on the current device.
 */
#ifndef SPSHELL_H
#define SPSHELL_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sp_shell sp_shell; /* opaque */

typedef enum {
    SP_OK = 0,
    SP_ERR_INVALID_ARG = 1, /* Nphi != 2 Ntheta, Nr < 2, Ntheta < 2, r_out <= r_in, r_in <= 0, L < 0, L > Ntheta-1,
                               null pointer, short workspace, rank > 3, malformed tensor descriptor */
    SP_ERR_NOT_BUILT = 2,   /* a hot call before sp_build_matrices */
    SP_ERR_ALLOC = 3,       /* host or device allocation failed */
    SP_ERR_CUDA = 4,        /* a CUDA runtime call or kernel launch failed */
    SP_ERR_UNSUPPORTED = 5, /* tensor index structure outside the supported set (see sp_tensor_desc) */
    SP_ERR_SCRATCH_LIMIT = 6 /* sp_tensor_filter_noalloc: the call needs more than SP_NOALLOC_SCRATCH_BYTES of scratch */
} sp_status;

/* Per-tensor index layout: the paper's d(u^mu) made explicit.
 * Stored components are the canonical multi-indices in row-major order over the indices, a
 * symmetric pair stored as its upper triangle; component c lives in state field `field[c]`.
 * A 4-dimensional index runs (t,x,y,z), its t value is a spin-0 spectator (reading Q17); a
 * 3-dimensional index runs (x,y,z).
 * Supported: rank 0; rank 1; rank 2 with sym = (0,1) and equal dims; rank 3 with sym = (1,2) and
 * equal dims on the pair (any first-index dim).  Anything else: SP_ERR_UNSUPPORTED. */
typedef struct {
    int rank;         /* 0..3 */
    int index_dim[3]; /* per index: 4 = spacetime (t,x,y,z), 3 = spatial (x,y,z); unused entries ignored */
    int sym_first;    /* indices of the one symmetric pair, or -1, -1 */
    int sym_second;
    const int *field; /* HOST pointer, length = number of stored components */
} sp_tensor_desc;

/* Create the shell descriptor (host only, no CUDA call).  PAPER.md:55-78 (eq. 2-5).
 * L = highest spherical-harmonic degree KEPT by the filter, 0 <= L <= Ntheta-1 (the paper's
 * n_f = Ntheta-1-L top degrees are removed). */
sp_status sp_shell_create(int Nr, int Ntheta, int Nphi, double r_in, double r_out, int L, sp_shell **out);
sp_status sp_shell_destroy(sp_shell *shell);

/* Build all matrices on the host in extended precision and upload them once (PAPER.md:114, 174, 180,
 * 215, 289, 374): CD^ (eq. 9), FD for 2 Ntheta and Nphi (eq. 8), the real Fourier analysis/synthesis
 * matrices (eq. 23-24, with B_jm = sin, reading Q1), and F^n_m = P f P^+ (eq. 48, 49, 62) for
 * n = -3..3, m = 0..L, built by the paper's own route: the n-recursion (42)-(44) (evaluated in
 * binary128) and the SVD pseudo-inverse.  Synchronous.  Without a CUDA device the host matrices are
 * still built (sp_get_matrix then works, so the host logic can be tested) but the call returns
 * SP_ERR_CUDA and every hot call keeps returning SP_ERR_NOT_BUILT.
 * SIZE LIMIT.  The gradient kernels keep an antipodal pair of (r, theta) planes of one field in one SM's shared memory:
 * shells with 2 * Ntheta8 * (Nr8 + 4) * 8 bytes plus the tables above 227 KB (Ntheta8, Nr8 = sizes rounded up to 8; e.g.
 * 129 x 128 x 256) return SP_ERR_UNSUPPORTED here.  The largest BASELINE grid, 65 x 96 x 192, uses 117 KB; the method
 * itself targets n <~ 100 per direction. */
sp_status sp_build_matrices(sp_shell *shell);

/* Workspace sizes in bytes for nfields fields (filter: nfields = total stored components of the
 * tensors passed).  Any pointer may be NULL. */
sp_status sp_workspace_bytes(const sp_shell *shell, int nfields, size_t *grad, size_t *filter, size_t *wave);

/* Cartesian gradient of nfields fields (eq. 6; 98-112 eq. 7-9; 142-166 eq. 13-19; 72).
 * u_dev: [nfields] state-shaped.  du_dev: [3][nfields] state-shaped = d/dx, d/dy, d/dz of every field
 * (du_dev[(c*nfields + mu)*Npts + point]).  du_dev must not overlap u_dev. */
sp_status sp_cartesian_gradient(const sp_shell *shell, const double *u_dev, int nfields, double *du_dev,
                                void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* Yn tensor filter (eq. 51-56, 60-62): dyad projection -> phi analysis (eq. 33) ->
 * per-(n,m) theta matrix (eq. 62) -> phi synthesis (eq. 31) -> recombination, for every radius.
 * u_dev, out_dev: [nfields] state-shaped; out_dev may equal u_dev.  Fields belonging to no tensor
 * are copied through unchanged.  A field may belong to at most one tensor. */
sp_status sp_tensor_filter(const sp_shell *shell, const double *u_dev, double *out_dev, int nfields,
                           const sp_tensor_desc *tensors, int ntensors,
                           void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* The same filter for callers that cannot allocate or pass a workspace (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): sp_tensor_filter with its scratch (the spin-weight components and the two coefficient arrays)
 * in a file-scope `static __device__` array of SP_NOALLOC_SCRATCH_BYTES = 32 MiB inside the library, which every GPU that loads
 * the library holds until the process exits.  Arguments, layout, results and errors as sp_tensor_filter, minus the workspace.
 *   - Allocates NOTHING on the device: no cudaMalloc / cudaFree / allocating library routine; the first call on a device resolves
 *     the array's device address once (cudaGetSymbolAddress, with that device current) -- make that first call outside a capture.
 *   - LIMIT: the call needs ncomp * (Nr Ntheta Nphi + 2 * roundup4(2L+1) * Nr Ntheta) * 8 bytes, ncomp = stored components of all
 *     tensors (the `filter` figure of sp_workspace_bytes(shell, ncomp, ...)): e.g. the 50-field GHG state at 17 x 24 x 48
 *     (20.9 MB) or the 5-field wave state at 33 x 64 x 128 (31.1 MB) fit, the GHG state at 33 x 48 x 96 (172 MB) does not.
 *     Beyond the limit the call launches nothing and returns SP_ERR_SCRATCH_LIMIT; use sp_tensor_filter with your own workspace.
 *   - SHARED: every call on a device uses the same array, which keeps the last call's contents.  Nothing in it has to start at
 *     zero (every region is written before it is read within a call), so nothing is cleared; but two calls that OVERLAP on the GPU
 *     (different streams, or concurrent host threads) race on it.  Calls on one stream, or ordered by events, are safe. */
#define SP_NOALLOC_SCRATCH_BYTES (32u * 1024u * 1024u)
sp_status sp_tensor_filter_noalloc(const sp_shell *shell, const double *u_dev, double *out_dev, int nfields,
                                   const sp_tensor_desc *tensors, int ntensors, void *cuda_stream);

/* First-order scalar wave RHS with characteristic boundaries (BASELINE.json config 5; W1-W3):
 * u = (psi, Pi, Phi_x, Phi_y, Phi_z);  d_t psi = -Pi, d_t Pi = -d_i Phi_i, d_t Phi_i = -d_i Pi; on the
 * shells k = 0 and k = Nr-1 the incoming characteristic field is frozen (A.16). */
sp_status sp_rhs_first_order_wave(const sp_shell *shell, const double *u_dev, double *dudt_dev,
                                  void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* ---- Generalized-harmonic (GHG) Einstein system, Appendix A ----
 * State u: 50 state-shaped fields, g_ab (tt,tx,ty,tz,xx,xy,xz,yy,yz,zz), k_ab (same ten; eq. A.6), d_iab (i = x,y,z
 * slowest, then the same ten).  H: gauge source H_a, 4 fields; dH: its Cartesian gradient, [3][4] fields (d_x H_t, d_x H_x,
 * ..., d_z H_z); d_t H_a = 0 (A.18).
 *
 * sp_rhs_ghg: dudt = right-hand side (A.8)-(A.10) with gamma0 = gamma2 = 1, gamma1 = -1, the dependent
 * quantities (lapse, shift, inverse metrics, Christoffel symbols, nabla_a H_b) by (A.3)-(A.5), (A.11) and PAPER.md:682; the
 * spatial derivatives of u are taken by sp_cartesian_gradient into the workspace.  bc_outer != 0: the freezing condition
 * (A.20)-(A.21) is applied on the outer shell k = Nr-1 (s_i = outward normal x_i/r normalised with gamma^{ij}).  All
 * pointers are device pointers owned by the caller; dudt must not alias u; workspace >= sp_ghg_workspace_bytes.
 * Asynchronous on cuda_stream, allocates nothing.  A metric that is not Lorentzian at some point gives NaN there (no check). */
sp_status sp_ghg_workspace_bytes(const sp_shell *shell, size_t *bytes);
sp_status sp_rhs_ghg(const sp_shell *shell, const double *u_dev, const double *H_dev, const double *dH_dev, double *dudt_dev,
                     int bc_outer, void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* Initial data from a metric with d_t g_ab = 0: on entry u holds g_ab (fields 0..9) and d_iab (fields
 * 20..49); fills k_ab = (beta^i/alpha) d_iab (A.6) into fields 10..19 and H_a = -Gamma_a (A.18) into H (4 fields). */
sp_status sp_ghg_init(const sp_shell *shell, double *u_dev, double *H_dev, void *cuda_stream);

/* Nested shells (PAPER.md:39, 616 name them as future work and specify nothing: DESIGN.md section 11).
 * sp_rhs_wave_shell is sp_rhs_first_order_wave with the boundary treatment chosen per boundary sphere: bc_inner / bc_outer = 1
 * applies the freezing condition (A.16) on k = 0 / k = Nr-1 (a physical boundary), 0 leaves the raw right-hand side there (an
 * interface with a neighbouring shell, to be coupled by sp_wave_interface).  Same arguments, workspace and errors otherwise. */
sp_status sp_rhs_wave_shell(const sp_shell *shell, const double *u_dev, double *dudt_dev, int bc_inner, int bc_outer,
                            void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* Characteristic coupling of two shells on their shared sphere r = inner.r_out = outer.r_in ((A.13)-(A.16) with
 * the zeroed incoming part replaced by the neighbour's): with n = r^, U+ = Pi + n.Phi (moving outward) is taken from the inner
 * shell's raw RHS row k = Nr_inner-1, U- = Pi - n.Phi (moving inward) from the outer shell's raw RHS row k = 0; BOTH rows get
 * d_t Pi = (U+ + U-)/2 and the normal part n.d_t Phi = (U+ - U-)/2; the tangential part of d_t Phi and d_t psi stay each shell's
 * own.  dudt_inner_dev / dudt_outer_dev: [5] state-shaped RHS arrays of the two shells (raw on the shared sphere), updated in
 * place.  The shells must share Ntheta and Nphi and the radius (SP_ERR_INVALID_ARG otherwise).  Asynchronous, allocates nothing. */
sp_status sp_wave_interface(const sp_shell *inner, double *dudt_inner_dev, const sp_shell *outer, double *dudt_outer_dev,
                            void *cuda_stream);

/* Time step of the method of lines, eq. (63) (reading W4): dt = lambda * min(dx) with min(dx) the
 * smaller of the first radial spacing r_1 - r_0 and the azimuthal spacing 2 r_0 sin(theta_0) sin(pi / Nphi) on the innermost
 * sphere next to the pole.  Host arithmetic on the shell's grid parameters; no device, no build needed.  lambda <= 0 is
 * SP_ERR_INVALID_ARG. */
sp_status sp_wave_dt(const sp_shell *shell, double lambda, double *dt_out);

/* Graded scalar filter Yg, eq. (59): component mu of the 50-field GHG state keeps the degrees l <= L + d(u^mu),
 * d = its number of spatial indices (g_tt: 0, g_tx: 1, g_xx: 2, ...; d_iab adds one), capped at the grid's Ntheta - 1.  Host only. */
sp_status sp_ghg_graded_degree(const sp_shell *shell, int field, int *L_out);

/* y <- a*x + b*y over n doubles (the RK4 combination steps of config 5). */
sp_status sp_axpby(double a, const double *x_dev, double b, double *y_dev, size_t n, void *cuda_stream);

/* One combination step of the classical RK4 scheme over n doubles, u and k read once:
 *     acc_out   = acc_in + c_acc * k
 *     stage_out = u + c_stage * k            (skipped when stage_out is NULL)
 * All pointers are device pointers owned by the caller.  acc_out may equal acc_in or u (the last stage writes the new
 * state over u); acc_in may equal u (the first stage).  stage_out must be distinct from every other array and acc_out
 * from k, else SP_ERR_INVALID_ARG.  Asynchronous on cuda_stream, allocates nothing. */
sp_status sp_rk4_stage(const double *u_dev, const double *k_dev, const double *acc_in_dev, double *acc_out_dev,
                       double *stage_out_dev, double c_acc, double c_stage, size_t n, void *cuda_stream);

/* Copy one host-built matrix out (for tests).  which: 0 = CD^ (Nr x Nr), 1 = FD_{2Ntheta} upper half
 * (Ntheta x 2Ntheta), 2 = FD_{Nphi} (Nphi x Nphi), 3 = Fourier analysis rows (2L+1 x Nphi; row 0 = a_0,
 * row 2m-1 = a_m, row 2m = b_m), 4 = Fourier synthesis (Nphi x 2L+1, same column order),
 * 5 = F^n_m (Ntheta x Ntheta; n in -3..3, m in 0..L).  Row-major into host_out (may be NULL to
 * query the shape). */
sp_status sp_get_matrix(const sp_shell *shell, int which, int n, int m, double *host_out, int *rows, int *cols);

/* Measure the FP64 issue peak of this device with a register-only DMMA (mode 0) or DFMA (mode 1)
 * loop; returns TFLOP/s.  Used by bench.py as the live denominator of the FP64 roofline. */
sp_status sp_probe_fp64_peak(int mode, double *tflops_out);

/* Per-stage device timing.  While enabled, the hot calls record CUDA events on the caller's stream
 * between their stages; sp_profile_read synchronises on them and returns the last call's durations in
 * milliseconds: ms7[0] d/dphi product, [1] d/dr + d/dtheta + chain rule, [2] dyad projection,
 * [3] phi analysis, [4] theta matrices, [5] phi synthesis, [6] recombination (-1 if not recorded). */
sp_status sp_profile_enable(sp_shell *shell, int on);
sp_status sp_profile_read(const sp_shell *shell, double *ms7_host);

/* Kernel variants sp_build_matrices selected for this shell (reporting only): out[0] = variant of the theta kernel chosen
 * by a timing run at build: NT + 20 * (rsplit - 1) with NT = 3 or 1 column tiles per warp and rsplit = 1 or 2 row blocks of
 * latitudes per (component, m, radial block), i.e. 3, 1, 23 or 21 (0 = generic kernel), out[1] = radial tiles per warp task of the
 * (r,theta) gradient kernel (3 or 5), out[2] = 1 if d/dphi uses the reflection-folded kernel, out[3] = 2 if the
 * double-buffered variant of the persistent (r,theta) kernel fits (it is used by calls with at least three waves of planes).  SP_ERR_NOT_BUILT before sp_build_matrices. */
sp_status sp_get_tuning(const sp_shell *shell, int out[4]);

/* Number of kernels the hot calls have launched since the library was loaded (host-side counter). */
unsigned long long sp_launch_count(void);

const char *sp_status_string(sp_status s);

#ifdef __cplusplus
}
#endif
#endif /* SPSHELL_H */
