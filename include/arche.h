/* arche.h -- C ABI of the B200-native hot path of Arche's orbital-free MD (arXiv 2606.13283):
 * finite-temperature Thomas-Fermi SCF on a periodic 3D grid + the per-MD-step ion-grid work.
 *
 * Citations: P:NNN = PAPER.md line NNN.  All computation behind these calls runs in hand-written
 * CUDA kernels for sm_100a in fp64 (own 3D FFT included); there is no CPU fallback.
 *
 * Conventions
 *   grid fields      real or complex (interleaved re,im) fp64, layout [z][y][x], x fastest
 *   reciprocal grid  k = (mx/Lx, my/Ly, mz/Lz), m in [-N/2+1, N/2], storage index i -> m = i (i<=N/2) else i-N
 *   transform        fhat(k) = dV sum_r f(r) exp(-2 pi i k.r);  f(r) = (1/|Omega|) sum_k fhat(k) exp(+2 pi i k.r)
 *   units            Hartree atomic units; positions in bohr, any value (periodic)
 *   pointers         "d_" = DEVICE pointer, "h_" = HOST pointer; the caller owns every array and the workspace
 *   errors           every call returns ARCHE_OK (0) or a negative code; nothing throws or aborts
 *   stream           all work is ordered on params.stream; calls that fill a host result synchronise that stream
 */
#ifndef ARCHE_H
#define ARCHE_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

#define ARCHE_OK 0
#define ARCHE_EINVAL (-1)   /* bad argument / call order */
#define ARCHE_ENOMEM (-2)   /* workspace too small */
#define ARCHE_ENOCONV (-3)  /* SCF hit scf_max_iter; the last iterate stays readable */
#define ARCHE_ENAN (-4)     /* non-finite value met */
#define ARCHE_ECUDA (-5)    /* CUDA runtime error (see arche_last_error) */

typedef struct arche_ctx arche_ctx; /* opaque, owned by the library */

typedef struct {
  double cell[3];        /* Lx, Ly, Lz in bohr, orthorhombic */
  int grid[3];           /* Nx, Ny, Nz; each 2^a 3^b, >= 4 and <= 1024 */
  int n_ions;            /* >= 0 */
  const double *h_Z;     /* [n_ions] valence charges, host, copied at init */
  const double *h_mass;  /* [n_ions] ion masses in electron masses, host, copied at init */
  double kT;             /* electron (= ion) temperature in Hartree */
  int xc;                /* 0: none (the paper's own TF derivations); 1: Perdew-Zunger 1981 LDA, constants as
                            printed (eps_c, V_c jump by ~3e-5 Ha at r_s = 1: stop rule of DESIGN.md reading A13);
                            2: the same with C, D at full precision from PZ's own continuity conditions at r_s = 1
                            (continuous eps_c and V_c, strict stop rule; reading A13b) */
  double psp_rc;         /* Ashcroft empty-core radius in bohr (BASELINE.json: 1.12) */
  int init_mode;         /* 0: uniform input density each step; 1: one-center profile */
  int mix_mode;          /* 0: fixed w; 1: More et al. w = U/(K+U) */
  double mix_w_fixed;    /* n_o = n_a + w (n_i - n_a); <= 0: automatic, the largest single-mode value
                            lambda/(1+lambda), lambda = chi0/(pi k_min^2) (reading A11d) */
  int mix_warmup;        /* SCF iterations run with mix_w_fixed before More's w is used */
  double scf_tol_F;      /* stop when |F_k - F_{k-1}| < scf_tol_F (Ha) ... */
  double scf_tol_dn;     /* ... and ||n_i - n_a||_L2 / ||n_a||_L2 < scf_tol_dn */
  int scf_max_iter;
  int scf_fixed_iter;    /* > 0: run exactly this many iterations (parity replay) */
  double ewald_alpha;    /* <= 0: automatic (reading A18) */
  double n_electrons;    /* <= 0: sum_j Z_j (neutral cell); > 0: that many electrons on a uniform background */
  int psp;               /* 0: Ashcroft empty core with psp_rc (BASELINE.json); 1: tabulated form factor (f2: the paper's
                            average-atom norm-conserving pseudopotential, or any other local potential) */
  int psp_nk;            /* psp = 1: table length (>= 4) */
  double psp_dk;         /* psp = 1: table spacing in k (1/bohr, ordinary frequency); (psp_nk-1) psp_dk must cover every
                            |k| of the grid, else ARCHE_EINVAL */
  const double *h_psp_table; /* psp = 1: HOST [psp_nk], copied at init: Du(k_m), k_m = m psp_dk -- the non-Coulomb part of the
                            form factor per unit charge, V_s(k) = Z_s (-1/(pi k^2) + Du(k)), interpolated by the cubic
                            Lagrange polynomial through the four nearest nodes (reading A22); Du(0) is the
                            k = 0 constant alpha_s/Z_s of Eq. 55 */
  double mix_mu_tol;     /* > 0: More's w is used only once two successive mu_a differ by <= mix_mu_tol kT (1 - w_prev) ("once the
                            chemical potential fluctuations are small"; latched; reading A11b); <= 0: off */
  double mix_chi_floor;  /* > 0: in K of Eq. 31 dn_a/dmu is bounded below by mix_chi_floor x its uniform-gas value chi_0: where
                            n_a underflows (chi -> 0) next to a finite n_i the quadratic model overstates the stiffness by
                            hundreds of orders of magnitude and w collapses to 0 (reading A11c); <= 0: Eq. 31 as
                            printed */
  int ensemble;          /* arche_md_step: 0 microcanonical, velocity Verlet; 1 isokinetic (ref. [48]; SURVEY.md 8
                            f4; reading A23): the half kicks are the exact constant-force flow of the Gaussian
                            isokinetic equations m dv/dt = F - alpha m v, alpha = sum F.v / sum m v^2, so the ion kinetic
                            energy of the initial velocities is conserved to round-off */
  void *d_workspace;     /* device memory, >= arche_workspace_bytes(), 256-byte aligned */
  size_t workspace_bytes;
  void *stream;          /* cudaStream_t (0 = default stream) */
} arche_params;

typedef struct {
  double mu;                                   /* chemical potential mu_a of Eq. 19 */
  double F_total;                              /* F0 + E_xc + E_H + E_ie + E_ie0 + U_ii (P:327-332 without K_i) */
  double F0, E_H, E_xc, E_ie, E_ie0, U_ii;
  double K_e, K_i;                             /* Eq. 38 and Eq. 36 */
  double dn_l2;                                /* ||n_i - n_a|| / ||n_a|| of the last iteration */
  double w_last, U_mix, K_mix;                 /* Eq. 30-31 */
  double tol_F_eff, tol_dn_eff;                /* the tolerances the stop rule applied in the last iteration (reading A13) */
  int scf_iters, mu_evals, converged;
  int flip_seen;                               /* 1: a PZ81 branch flip was detected and the tolerances were widened (A13) */
  int F_evals;                                 /* iterations of the solve that evaluated the free energy: all of them in the
                                                  split form, in parity replays and with xc = 1; under the stop rule with
                                                  xc = 0 / 2 only those where the rule can use it (the last two or so:
                                                  the paper's own criterion P:231 needs no F; ARCHE_LAZY_F=0 disables) */
} arche_result;

/* Bytes of device workspace arche_scf_init will carve up for these parameters (0 on bad parameters). */
size_t arche_workspace_bytes(const arche_params *p);

/* Validate, copy Z/mass, build twiddle tables and reciprocal-space factors on the device (they depend only on
 * cell/grid/T).  *out is set on success; destroy with arche_destroy.  No device allocation happens after init. */
int arche_scf_init(const arche_params *p, arche_ctx **out);
void arche_destroy(arche_ctx *c);
const char *arche_last_error(const arche_ctx *c);

/* One SCF solve for ion positions d_pos[n_ions*3] (row-major [ion][xyz]):
 * structure factor S_Z(k), ionic potential Vhat_ie, Ewald, input density
 * (uniform or Eq. 20), then SCF iterations with mixing until the stop rule;
 * finally stores ghat = nhat/S_Z.  *h_out filled after a stream synchronise. */
int arche_scf_solve(arche_ctx *c, const double *d_pos, arche_result *h_out);

/* Split form of the solve (used for step-by-step parity and for timing single iterations):
 * begin = per-step ion-grid work + input density; iter = exactly one SCF iteration. */
int arche_scf_begin(arche_ctx *c, const double *d_pos);
int arche_scf_iter(arche_ctx *c, arche_result *h_out);
/* Replace the input density n_i (d_n: [Nz][Ny][Nx] real, device); nhat_i is recomputed by the FFT. */
int arche_set_input_density(arche_ctx *c, const double *d_n);

/* Total force F^ie (Eq. 56) + F^ii (Eq. 45-47) on every ion from the last active density,
 * written to d_F[n_ions*3].  ARCHE_EINVAL before any solve. */
int arche_forces(arche_ctx *c, double *d_F);

/* Average virial stress tensor and pressure of the last solve (Eq. 34-35; terms Eq. 37
 * P:355, Eq. 39, Eq. 48-51, Eq. 54, sigma^ie P:483-487; sign convention and the LDA term:
 * DESIGN.md reading A21): sigma_mn = (1/|Omega|) dE/d(eps_mn) at fixed scaled coordinates and fixed Ewald alpha,
 * P = -tr(Sigma)/3, Hartree/bohr^3.
 * h_out: HOST array of ARCHE_STRESS_DOUBLES doubles, owned by the caller: 9 rows (i, e, xc, pp, pm, je, ee, ie,
 * total) x 6 columns (xx, yy, zz, yz, xz, xy), then P.  d_vel: DEVICE [n_ions*3] ion velocities for sigma^i, or NULL
 * (sigma^i = 0).  Stream-ordered, synchronises before filling h_out.  ARCHE_EINVAL before any solve. */
#define ARCHE_STRESS_DOUBLES 55
int arche_stress(arche_ctx *c, const double *d_vel, double *h_out);

/* Change the iteration control of the following solves: scf_max_iter (0 keeps the current value) and scf_fixed_iter
 * (> 0: run exactly that many iterations -- parity replay of an oracle run solve by solve; 0: stop rule). */
int arche_set_scf_iterations(arche_ctx *c, int scf_max_iter, int scf_fixed_iter);

/* One velocity-Verlet step of length dt (a.u.) (reading D2): half kick, drift, SCF solve at the
 * new positions, forces, half kick (params.ensemble = 1: isokinetic half kicks, same splitting).  d_pos/d_vel [n_ions*3] are updated in place.  The first call also solves
 * at the starting positions to obtain the initial forces.  Later calls reuse the forces of the previous step: a caller
 * that edits the positions between two steps must call arche_scf_solve + arche_forces on them first.
 * Returns ARCHE_ENOCONV when either solve of the step hit scf_max_iter (the step is still taken). */
int arche_md_step(arche_ctx *c, double dt, double *d_pos, double *d_vel, arche_result *h_out);
/* Same step through HOST buffers: positions/velocities are copied in, the step runs, positions, velocities and
 * forces (h_F may be NULL) are copied back -- the paper's per-step host<->device traffic. */
int arche_md_step_host(arche_ctx *c, double dt, double *h_pos, double *h_vel, double *h_F, arche_result *h_out);

/* Field read-back for parity tests (device destination buffers).
 * real   which: 0 n_a (active density of the last iteration), 1 n_i (next input density), 2 V_i
 * complex which: 0 nhat_a, 1 Vhat_ie, 2 S_Z, 3 ghat, 4 nhat_i */
int arche_get_real(arche_ctx *c, int which, double *d_dst);
int arche_get_complex(arche_ctx *c, int which, double *d_dst);
int arche_get_density(arche_ctx *c, double *d_n); /* = arche_get_real(c, 0, d_n) */

/* Stand-alone entry points of individual kernels (unit parity + roofline benches). */
/* 3D complex FFT, unnormalised, out-of-place or in-place (d_in == d_out allowed); sign = -1 forward, +1 inverse.
 * d_scratch: 16*Nx*Ny*Nz bytes. */
int arche_fft3d(arche_ctx *c, const double *d_in, double *d_out, double *d_scratch, int sign);
/* The same transform for callers that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): no d_scratch argument, no cudaMalloc / cudaFree / allocating library call inside.  The scratch is a
 * file-scope `static __device__` array of ARCHE_FFT3D_STATIC_MAX_POINTS complex doubles (4 MiB) in the library image:
 * every GPU that loads the library holds it until exit.  Grids with Nx*Ny*Nz > ARCHE_FFT3D_STATIC_MAX_POINTS are rejected
 * with ARCHE_EINVAL and a message in arche_last_error.  d_in / d_out: device pointers, 16*Nx*Ny*Nz bytes each, caller
 * owned, d_in == d_out allowed.  Results are bit-identical to arche_fft3d.  ALL calls on one GPU (any context, any
 * stream) share the one array and it keeps the last call's contents: nothing in it needs clearing (the first pass
 * overwrites every element before it is read), but two calls that overlap on the GPU -- different streams, different
 * contexts or processes' threads on the same device without ordering -- race on it.  Serialise them. */
#define ARCHE_FFT3D_STATIC_MAX_POINTS (64 * 64 * 64)
int arche_fft3d_static(arche_ctx *c, const double *d_in, double *d_out, int sign);
/* f4 (grids beyond one GPU): the complex transform of arche_fft3d decomposed into slabs
 * over n_ranks GPUs (one process per GPU, or several slabs on one GPU), unnormalised, same sign convention.
 * Layouts: "z slab" of rank r = planes r Nz/R ... (r+1) Nz/R - 1 of the field, [Nz/R][Ny][Nx]; "y slab" of rank r = rows
 * r Ny/R ... of every plane, [Nz][Ny/R][Nx].  sign = -1 maps z slabs (real space) to y slabs (reciprocal space,
 * transposed output); sign = +1 maps y slabs back to z slabs.  Ny and Nz must be multiples of n_ranks <= 16.
 * The transpose is not a separate exchange: the pass before it stores every element straight into the slab of the
 * rank that owns it afterwards -- h_peer[q] is the DEVICE address, valid on the calling GPU, of rank q's destination
 * slab (its y slab for sign = -1, its z slab for sign = +1): peer memory mapped over NVLink (arche_ipc_open, or
 * cudaDeviceEnablePeerAccess within a process) or a local buffer.  h_peer itself is a HOST array of n_ranks pointers.
 *   arche_fft3d_slab_scatter: sign = -1: x and y passes on the z slab d_in (d_scratch: 16 Nx Ny Nz/R bytes, device), the
 *     y pass scattering into the peers' y slabs; sign = +1: z pass on the y slab d_in scattering into the peers' z slabs
 *     (d_scratch unused, may be NULL).  d_in is not modified.
 *   -- every rank's scatter must have completed (stream synchronise + a barrier across the ranks) --
 *   arche_fft3d_slab_finish: sign = -1: z pass in place on this rank's y slab; sign = +1: y and x passes in place on this
 *     rank's z slab.
 * Both are stream-ordered on the context's stream and allocate nothing.  The context supplies the axis plans of the
 * GLOBAL grid (its SCF arrays are not touched). */
int arche_fft3d_slab_scatter(arche_ctx *c, const double *d_in, double *d_scratch, double *const *h_peer, int n_ranks,
                             int rank, int sign);
int arche_fft3d_slab_finish(arche_ctx *c, double *d_slab, int n_ranks, int sign);
/* Slab buffers that another process can map: arche_slab_alloc is a plain cudaMalloc on the current device (an IPC
 * handle names a whole allocation, so such buffers must not come from a caching allocator's pool); arche_ipc_export
 * writes the 64-byte handle of such a buffer to HOST memory, arche_ipc_open maps a peer's buffer into this process
 * (peer access enabled lazily) and returns its device address here, arche_ipc_close unmaps it. */
int arche_slab_alloc(size_t bytes, void **d_out);
int arche_slab_free(void *d_ptr);
int arche_ipc_export(const void *d_ptr, unsigned char *h_handle64);
int arche_ipc_open(const unsigned char *h_handle64, void **d_out);
int arche_ipc_close(void *d_ptr);
/* The transform pair the SCF itself uses: real field [Nz][Ny][Nx] <-> half spectrum, through the r2c / c2r x passes and
 * the y/z passes (register two-stage kernels for N in {32,64,128,192,256,384}, generic radix kernels otherwise).
 * forward: d_full_out receives the full unnormalised spectrum [Nz][Ny][Nx] complex (the stored half expanded by
 * Hermitian symmetry); inverse: d_full_in must be Hermitian (only ix <= Nx/2 is read), d_real_out receives the
 * unnormalised inverse transform.  Both use the context's FFT scratch array. */
int arche_rfft3d_forward(arche_ctx *c, const double *d_real_in, double *d_full_out);
int arche_rfft3d_inverse(arche_ctx *c, const double *d_full_in, double *d_real_out);
/* I_j(eta) for twice_j in {-1,1,3} on n device values */
int arche_fermi_dirac(arche_ctx *c, int twice_j, const double *d_eta, double *d_out, size_t n);
/* number of kernels this context has launched so far (for bench.py's gpu_launches) */
long long arche_launch_count(const arche_ctx *c);

/* Per-kernel-class timing with CUDA events on params.stream (adds ~2 event records per launch; off by default).
 * Classes: 0 inverse-FFT z pass with the G-space potential prologue (S1), 1 FFT y passes, 2 inverse-FFT x pass with
 * the V_i epilogue (S2), 3 mu passes (S3), 4 density kernel (S4), 5 forward-FFT x pass reading the real n_a,
 * 6 forward-FFT z pass with the G-space reductions (S5), 7 mixing (S6), 8 structure factor (P1,P2), 9 force sum (P5),
 * 10 Ewald pair kernel, 11 other.  On grids beyond the L2 the pointwise work runs as streaming kernels around plain
 * passes (arche_is_fused() == 0): 12 G-space potential assembly + mixing (S1/S6), 13 V_i assembly + XC + first mu
 * evaluation (S2), 14 density and local reductions (S4), 15 G-space reductions (S5); classes 0, 2, 5, 6 are then the
 * plain passes and 4 is unused.  16 field sums of arche_stress (f1).  arche_profile_get returns the summed milliseconds and launch count of a class. */
int arche_profile_enable(arche_ctx *c, int on);
int arche_is_fused(const arche_ctx *c);
/* 1 when arche_scf_solve runs the whole SCF loop in one persistent cooperative launch (fused form on 32^3 / 64^3 grids;
 * the profile classes 0-6 then receive the phase times block 0 measures with %globaltimer) */
int arche_is_persistent(const arche_ctx *c);
int arche_profile_get(arche_ctx *c, int cls, double *h_ms_total, long long *h_launches);

/* Measured rooflines for the fractions bench.py reports (peak_kernels.cuh): the fp64 FMA rate of the
 * vector pipe -- independent dependent-FMA chains on every SM, launched back to back for `seconds` (>= 1 for a
 * sustained figure); h_tflops[0] = sustained over the whole run, h_tflops[1] = best single launch; *h_ms (optional) = the
 * time it ran -- and the L2 read bandwidth in GB/s of a <= 32 MiB slice of the workspace swept 64 times. */
int arche_peak_fp64(arche_ctx *c, double seconds, double *h_tflops /*[2]*/, double *h_ms);
int arche_peak_l2(arche_ctx *c, double *h_gbs);

#ifdef __cplusplus
}
#endif
#endif
