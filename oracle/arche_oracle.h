/* CPU ORACLE -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, obviously-correct fp64 implementation of the finite-temperature Thomas-Fermi SCF
 * hot path of PAPER.md (arXiv 2606.13283, "Arche"), written from the paper.  It shares no code,
 * tables or headers with the CUDA path in paper_2606_13283_b200/.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
 *
 * Every host pointer is owned by the caller.  All arrays are row-major; grid fields are
 * [z][y][x] with x fastest; complex = interleaved (re, im) doubles (C99 double complex).
 *
 * Conventions: k = (mx/Lx, my/Ly, mz/Lz) with m in [-N/2+1, N/2]
 * (PAPER.md:142), storage index i -> m = i (i <= N/2) else i-N;
 * fhat(k) = dV * sum_r f(r) exp(-2 pi i k.r),  f(r) = (1/|Omega|) sum_k fhat(k) exp(+2 pi i k.r)
 * (PAPER.md:144-149 discretised so that both lines of Eq. 53, agree).
 *
 * Parity pins: tests/test_oracle_pins.py (every function below is pinned there except the SCF
 * iteration count / w history, which are "parity unpinned": they depend on DESIGN.md readings).
 */
#ifndef ARCHE_ORACLE_H
#define ARCHE_ORACLE_H
#ifdef __cplusplus
extern "C" {
#endif

typedef struct oracle_ctx oracle_ctx;

typedef struct {
  double cell[3];      /* Lx, Ly, Lz (bohr) */
  int grid[3];         /* Nx, Ny, Nz */
  int n_ions;
  const double *Z;     /* [n_ions] valence charges */
  const double *mass;  /* [n_ions] electron masses */
  double kT;           /* Hartree */
  int xc;              /* 0 none (paper's TF-only derivations), 1 PZ81 LDA as printed, 2 PZ81 with C, D
                          at full precision from its own continuity conditions at r_s = 1 (reading A13b) */
  double psp_rc;       /* Ashcroft empty-core radius (bohr) */
  int init_mode;       /* 0 uniform density every step, 1 one-center profile */
  int mix_mode;        /* 0 fixed w, 1 More et al. w = U/(K+U) */
  double mix_w_fixed;  /* n_o = n_a + w (n_i - n_a); <=0: lambda/(1+lambda), lambda = chi0/(pi k_min^2) (reading A11d) */
  int mix_warmup;      /* iterations with the fixed w before More's w */
  double scf_tol_F;    /* Ha */
  double scf_tol_dn;   /* relative L2 */
  int scf_max_iter;
  int scf_fixed_iter;  /* >0: run exactly this many iterations */
  double ewald_alpha;  /* <=0: auto */
  double n_electrons;  /* <=0: sum_j Z_j (neutral cell); >0: that many electrons on a
                          uniform neutralising background (uniform-gas and linear-response pins) */
  double mix_mu_tol;   /* >0: More's w only once |mu_k - mu_{k-1}| <= mix_mu_tol kT (1 - w_prev) (reading A11b) */
  int psp;             /* 0 Ashcroft empty core (psp_rc); 1 tabulated form factor (f2) */
  int psp_nk;          /* table length */
  double psp_dk;       /* table spacing in k (1/bohr, ordinary frequency) */
  double mix_chi_floor; /* >0: lower bound of dn_a/dmu in K (Eq. 31) in units of the uniform-gas value (reading A11c) */
  const double *psp_table; /* [psp_nk] Du(k_m): non-Coulomb part of the form factor per unit charge, u = -1/(pi k^2) + Du */
  int ensemble;        /* 0 microcanonical: velocity Verlet; 1 isokinetic: the ion kinetic energy is a
                          constant of the motion ("the isokinetic ensemble algorithm ... follows similar
                          lines [48]"; reading A23) */
} oracle_params;

typedef struct {
  double mu, F_total, F0, E_H, E_xc, E_ie, E_ie0, U_ii, K_e, K_i, dn_l2, w_last, U_mix, K_mix;
  double tol_F_eff, tol_dn_eff; /* tolerances the stop rule applied (reading A13) */
  int scf_iters, mu_evals, converged;
  int flip_seen;                /* a PZ81 branch flip was detected in this solve (reading A13) */
} oracle_result;

/* --- primitives ------------------------------------------------------------------------ */
/* I_j(eta) = int_0^inf t^j/(exp(t-eta)+1) dt, j = twice_j/2 in {-1/2,1/2,3/2} */
double oracle_fd(int twice_j, double eta);
double oracle_fd_half_inverse(double y);             /* eta with I_{1/2}(eta) = y */
/* unnormalised DFT along all three axes, in place; sign=-1: exp(-2 pi i mn/N), +1: exp(+...) */
void oracle_fft3d(int nx, int ny, int nz, double *a_complex, int sign);
void oracle_dft3d_naive(int nx, int ny, int nz, double *a_complex, int sign);
/* xc=1: Perdew-Zunger 1981 LDA, unpolarised: energy per electron and potential; xc=2: continuous variant (A13b) */
void oracle_xc(int xc, double n, double *eps_xc, double *v_xc);
/* S_Z(k) = sum_j Z_j exp(-2 pi i k.r_j) on the grid */
void oracle_structure_factor(const double cell[3], const int grid[3], int n_ions,
                             const double *pos, const double *Z, double *S_complex);
/* cubic Lagrange interpolation of a uniform table (f2; reading A22); du_dk may be NULL */
double oracle_table_interp(int nk, double dk, const double *tab, double k, double *du_dk);
/* Ashcroft empty-core form factor per unit charge: -cos(2 pi k rc)/(pi k^2), 0 at k=0 */
double oracle_vps_unit(double kabs, double rc);
double oracle_ewald_alpha(const double cell[3], const int grid[3]);
/* Ewald: U[0]=U_pp, U[1]=U_pm (incl. self term), U[2]=U_je; F[n_ions*3] = F_pp + F_pm */
void oracle_ewald(const double cell[3], const int grid[3], int n_ions, const double *pos,
                  const double *Z, double alpha, double U[3], double *F);

/* --- SCF / MD context -------------------------------------------------------------------- */
int oracle_init(const oracle_params *p, oracle_ctx **out);
void oracle_destroy(oracle_ctx *c);
/* per-MD-step ion-grid work + input-density initialisation for positions pos[n_ions*3] */
int oracle_scf_begin(oracle_ctx *c, const double *pos);
/* supply the one-center profile ghat [Nz][Ny][Nx] complex directly (pin of the clip/renormalise rule
 * of DESIGN.md reading A10); the next oracle_scf_begin with init_mode = 1 starts from S_Z ghat (Eq. 20) */
int oracle_set_profile(oracle_ctx *c, const double *ghat_complex);
/* supply the input density explicitly (real field); n_hat_i is recomputed by FFT */
int oracle_set_input_density(oracle_ctx *c, const double *n_i);
/* one SCF iteration (PAPER.md:217-231 + 257-311) from the current input density */
int oracle_scf_iter(oracle_ctx *c, oracle_result *out);
int oracle_scf_solve(oracle_ctx *c, const double *pos, oracle_result *out);
/* total force F^ie + F^ii on every ion from the last active density */
int oracle_forces(oracle_ctx *c, double *F);
/* Gaussian isokinetic half step (ref. [48]; reading A23): the exact flow over a time t of
 * m_j dv_j/dt = F_j - alpha m_j v_j, alpha = sum F.v / sum m v^2, for forces held constant; vel updated in place. */
void oracle_isokinetic_kick(int n_ions, const double *mass, const double *F, double t, double *vel);
/* one velocity-Verlet step (reading D2); ensemble = 1: the same splitting with the isokinetic
 * kick in place of the free one */
int oracle_md_step(oracle_ctx *c, double dt, double *pos, double *vel, oracle_result *out);
/* field access: which = 0 n_a, 1 n_i (next input), 2 V_i ; complex: 0 nhat_a, 1 Vhat_ie, 2 S_Z, 3 ghat, 4 nhat_i */
int oracle_get_real(oracle_ctx *c, int which, double *dst);
int oracle_get_complex(oracle_ctx *c, int which, double *dst);
/* F^ie only, for an arbitrary density given in G-space (used by the fixed-density FD pin) */
void oracle_force_ie(const double cell[3], const int grid[3], int n_ions, const double *pos,
                     const double *Z, double rc, const double *nhat_complex, double *F);
/* f1: average virial stress tensor and pressure from the last solve (PAPER.md:341-347 Eq. 34-35, :355 Eq. 37,
 * :372 Eq. 39, :423-440 Eq. 48-51, :458-461 Eq. 54, :483-487; LDA term: DESIGN.md reading A21).
 * sigma_mn = (1/|Omega|) dE/d(eps_mn) at fixed scaled coordinates and fixed Ewald alpha; P = -tr(Sigma)/3.
 * out[9*6 + 1]: rows i, e, xc, pp, pm, je, ee, ie, total; columns xx, yy, zz, yz, xz, xy; out[54] = P.
 * vel[n_ions*3] may be NULL (sigma^i = 0).  Pins: tests/test_oracle_stress_pins.py. */
#define ORACLE_STRESS_DOUBLES 55
int oracle_stress(oracle_ctx *c, const double *vel, double *out);
int oracle_num_threads(void);

/* --- f2: average-atom norm-conserving pseudopotential (aa_pseudopotential.c; Eq. 16-18) ---------- */
/* I_j(eta) for any eta (Sommerfeld expansion beyond eta = 500, 0 below -600) and the inverse of I_{1/2} built on it */
double oracle_fd_wide(int twice_j, double eta);
double oracle_fd_half_inverse_wide(double y);
/* Radial grid r_i = (i h)^2, i = 0..n-1 (n odd), h = sqrt(r_ws)/(n-1); all arrays [n], caller-owned. */
/* finite-T Thomas-Fermi average atom: nucleus Z in a neutral sphere of radius r_ws; fills r, n_aa (n_aa[0] = 0 stands for
 * the integrable r^(-3/2) singularity), *mu; returns 0 when converged */
int oracle_aa_solve(double Z, double r_ws, double kT, int xc, int n, double *r, double *n_aa, double *mu, int *iters);
/* Eq. 16-17 with r_cut = r[ic]: n_ps[n], abc = {a, b, c} */
int oracle_aa_pseudize(int n, const double *r, const double *n_aa, int ic, double *n_ps, double abc[3]);
/* Eq. 18 for any density of the sphere: V_ext[n]; n0lim = lim r^(3/2) dens (0 for a regular density) */
int oracle_aa_invert(double kT, int xc, int n, const double *r, const double *dens, double n0lim, double mu, double *V_ext);
/* out[m] = int_0^{r[ic]} f(r) 4 pi r^2 sin(2 pi k_m r)/(2 pi k_m r) dr */
void oracle_radial_ft(int n, const double *r, const double *f, int ic, int nk, const double *k, double *out);
/* out = {K_e, E_ext, E_H, E_xc} of a density in the sphere; V_ext == NULL: the Coulomb potential -Zc/r */
int oracle_aa_energy(double kT, int xc, int n, const double *r, const double *dens, double n0lim, const double *V_ext,
                     double Zc, double out[4]);

#ifdef __cplusplus
}
#endif
#endif
