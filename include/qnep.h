/*
 * qnep.h -- C ABI of the B200-native qNEP force evaluation (arXiv 2601.19034).
 *
 * One call, qnep_compute(), evaluates for given positions, species and a periodic cell of any
 * shape (orthorhombic or triclinic, PAPER.md :104) the total energy (Eq. 4), forces (Eq. 11),
 * total virial (Eq. 12 + Eq. 22), the neutralised partial charges (Eq. 1 second output node,
 * Eq. 33) and, on request, the per-ion Born effective charge tensor (Eq. 28).  Beside it:
 * qnep_compute_atom_virial (per-atom virial, Eq. 12 / 20 / 39), qnep_compute_host (host buffers),
 * qnep_md_run (velocity-Verlet driver, optionally with virial and charges every step),
 * qnep_response (Eq. 29-30), qnep_set_zbl (optional ZBL core), NEP4's 4-/5-body descriptors
 * (qnep_model_desc.l_max_4b / l_max_5b), the Ewald / PPPM selector, and
 * qnep_neutralise_noalloc (Eq. 33 for callers that may not allocate device memory).  Every step
 * runs in hand-written CUDA kernels for sm_100a inside this library; there is no CPU fallback,
 * no cuFFT and no other library on the path.
 *
 * Conventions
 *   - every function returns QNEP_OK (0) or a negative QNEP_ERR_* code; no C++ exception
 *     crosses this boundary; on error the outputs are unspecified but nothing is written
 *     out of bounds;
 *   - "_dev" pointers are DEVICE pointers owned by the caller (e.g. PyTorch tensors);
 *     "_host" pointers are HOST pointers owned by the caller and copied during the call;
 *   - the handle owns its workspace and its copy of the model; all work is enqueued on the
 *     caller's stream; qnep_compute() does not synchronise -- neighbour-capacity overflow
 *     and skin violation are detected on the device and reported by the NEXT call on the
 *     handle or by qnep_check() (which synchronises the stream);
 *   - units: Angstrom, eV, elementary charge; 1/(4 pi eps0) = 14.3996454784 eV A / e^2.
 */
#ifndef QNEP_H
#define QNEP_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct qnep_handle qnep_handle; /* opaque */

/*
 * Version of this boundary: raised whenever a struct below changes size or layout or an entry point changes its signature
 * (1: round-1 header; 2: qnep_model_desc grew by l_max_4b, l_max_5b; 3: qnep_neutralise_noalloc, qnep_abi_version).  The structs
 * carry no size field, so a caller built against another header would hand qnep_create a struct of the wrong size: compare
 * qnep_abi_version() (what the loaded library was built with) with QNEP_ABI_VERSION (what the caller was compiled with)
 * once after loading.  Needs no device.
 */
#define QNEP_ABI_VERSION 3
int qnep_abi_version(void);

enum {
    QNEP_OK = 0,
    QNEP_ERR_INVALID_ARG = -1,
    QNEP_ERR_UNSUPPORTED = -2,       /* order != 5, non-power-of-2 grid, > 4 species, cell narrower than r_c + skin      */
    QNEP_ERR_NEIGHBOR_OVERFLOW = -3, /* a neighbour list exceeded its capacity; capacity has been grown, call again */
    QNEP_ERR_SKIN_VIOLATED = -4,     /* an atom moved more than skin/2 since the last neighbour build */
    QNEP_ERR_CUDA = -5,
    QNEP_ERR_OOM = -6
};

/* The qNEP model (PAPER.md :37-60, Eq. 1; descriptor form: DESIGN.md reading S1-S5). Plain data, copied at create. */
typedef struct {
    int32_t n_types;      /* number of species T (1..4)                                                      */
    /* The next five describe the parameter vector; THIS VERSION accepts exactly n_max_r = n_max_a = 4, l_max = 4,
     * basis_r = basis_a = 8 (the shape of every BASELINE.json config; the kernels are specialised for it) and
     * qnep_create returns QNEP_ERR_UNSUPPORTED for anything else. */
    int32_t n_max_r;      /* radial descriptors  n = 0..n_max_r                                              */
    int32_t n_max_a;      /* angular descriptors n = 0..n_max_a                                              */
    int32_t l_max;        /* angular momentum l = 1..l_max                                                   */
    int32_t basis_r;      /* Chebyshev basis k = 0..basis_r (radial)                                         */
    int32_t basis_a;      /* Chebyshev basis k = 0..basis_a (angular)                                        */
    int32_t n_neurons;    /* hidden layer width N_neu (Eq. 1)                                                */
    double rc_r, rc_a;    /* radial / angular cutoff, Angstrom; rc_a <= rc_r; rc_r is also the real-space
                             Coulomb cutoff (:89-91)                                                         */
    int32_t mode;         /* 1: U^ES = U^r + U^k + U^s (Eq. 3); 2: U^ES = U^k (Eq. 5)                        */
    double sqrt_eps_inf;  /* Eq. 24, used only by the Born effective charges                                 */
    double q_total;       /* target total charge Q of Eq. 33                                                 */
    /* NEP4's higher-body angular terms (PAPER.md :39 defers to the NEP papers; reading Z2), one descriptor per
     * angular radial channel n each, appended behind the 3-body block: 4-body q_n = tr(T_n^3) with the l = 2 moment tensor
     * T_n = sum_j g_n(r_ij) (rhat rhat^T - 1/3), 5-body q_n = (w_n . w_n)^2 with w_n = sum_j g_n(r_ij) rhat.
     * THIS VERSION accepts (l_max_4b, l_max_5b) = (0, 0) [off] or (2, 1) [both on]; anything else: UNSUPPORTED.            */
    int32_t l_max_4b;
    int32_t l_max_5b;
} qnep_model_desc;

/* Reciprocal-space method -- the Ewald / PPPM selector (PAPER.md II.B.2 and II.F). */
typedef struct {
    int32_t method;       /* 0: no electrostatics; 1: Ewald summation (Eq. 7-9); 2: PPPM (Eq. 34-38)         */
    double alpha;         /* Ewald splitting parameter, 1/Angstrom; <= 0 selects pi / rc_r (:91)             */
    int32_t ewald_nmax2;  /* Ewald: keep integer n.n <= nmax2 (k = 2 pi n / L); <= 0 selects |k| <= 2 pi alpha (:110) */
    int32_t grid[3];      /* PPPM mesh N_x, N_y, N_z: powers of two, 16..512                                 */
    int32_t order;        /* PPPM interpolation order P; 5 only (:280)                                       */
} qnep_es_desc;

/* bit flags of `want` */
enum { QNEP_WANT_ENERGY = 1, QNEP_WANT_FORCES = 2, QNEP_WANT_VIRIAL = 4, QNEP_WANT_CHARGES = 8, QNEP_WANT_BEC = 16,
       QNEP_WANT_ATOM_VIRIAL = 32 /* qnep_compute_atom_virial only */ };

/* stages reported by qnep_get_timings (milliseconds of the last qnep_compute) */
enum {
    QNEP_T_NEIGHBOR = 0,   /* a1  cell list + neighbour lists (0 when not rebuilt)   */
    QNEP_T_PREP,           /*     cell-relative fp32 coordinates, skin check         */
    QNEP_T_DESC_RADIAL,    /* a2  skin-list walk: exact lists of the step + radial   */
    QNEP_T_DESC_ANGULAR,   /* a3                                                     */
    QNEP_T_NN,             /* a4, a5 (+ dU/dD, dq/dD of a10)                         */
    QNEP_T_REALSPACE,      /* a6, a8                                                 */
    QNEP_T_RECIPROCAL,     /* a7E or a7P-1..5, a9 (potential assembly)               */
    QNEP_T_FORCE_ANGULAR,  /* a10 (Fp combine) + a11 (angular partial forces)        */
    QNEP_T_FORCE_RADIAL,   /* a11 (radial partial forces, assembly, outputs)         */
    QNEP_T_BEC,            /* a12                                                    */
    QNEP_T_TOTAL,
    QNEP_T_COUNT
};

/* per-stage intermediates for the parity tests (qnep_debug_copy) */
enum {
    QNEP_DBG_DESCRIPTORS = 0, /* [N][n_desc] unscaled D^i, row per atom       */
    QNEP_DBG_SITE_ENERGY,     /* [N] U_i                                        */
    QNEP_DBG_Q_RAW,           /* [N] q_i before Eq. 33                          */
    QNEP_DBG_PHI,             /* [N] dU^ES/dq_i before the mean subtraction     */
    QNEP_DBG_FP,              /* [N][n_desc] dU_i/dD + phi_eff dq_i/dD          */
    QNEP_DBG_MESH_RHO,        /* [Nx][Ny][Nz] PPPM charge mesh                  */
    QNEP_DBG_F_STATIC,        /* [3][N] static electrostatic force              */
    QNEP_DBG_ENERGY_PARTS     /* [4] U^NEP, U^r, U^k, U^s                       */
};

/*
 * qnep_create: build a handle.
 *   params_host [n_params] float32, order:
 *     c_R[ti][tj][n][k], c_A[ti][tj][n][k], s[n_desc],
 *     then per type: w0[H][n_desc], b0[H], w1U[H], w1q[H]; then b1U, b1q.
 *   n_desc = (n_max_r + 1) + (n_max_a + 1) * l_max  [+ 2 (n_max_a + 1) with the 4-/5-body terms: 4-body block, then 5-body
 *   block].  The vector is copied.
 * Errors: INVALID_ARG (null pointer, wrong n_params, rc_a > rc_r), UNSUPPORTED, CUDA, OOM.
 */
int qnep_create(const qnep_model_desc *model, const float *params_host, size_t n_params,
                const qnep_es_desc *es, qnep_handle **out);

/* the Ewald / PPPM selector; may be called between computes.  Errors: INVALID_ARG, UNSUPPORTED. */
int qnep_set_electrostatics(qnep_handle *h, const qnep_es_desc *es);

/*
 * Neighbour policy: the cell list and the skin list (every pair within rc_r + skin) are rebuilt every
 * `rebuild_every` calls (0 or 1: every call).  Every call derives the exact lists (r < rc_r, r < rc_a) of
 * its own positions from the skin list, so results do not depend on skin.  Default: skin = 0, rebuild every call.
 */
int qnep_set_neighbor_policy(qnep_handle *h, double skin, int32_t rebuild_every);

/* Override the automatic list capacities (entries per atom, rounded up to a multiple of 4): cap_radial sizes the skin
 * list and the live radial list, cap_angular the live angular list; <= 0 keeps the automatic value (1.5 x the count
 * expected from the mean density + 24).  When a list overflows, the call that notices it returns
 * QNEP_ERR_NEIGHBOR_OVERFLOW, the handle drops an explicit capacity that proved too small and remembers the observed
 * count as a lower bound for its automatic sizing: the caller repeats the call. */
int qnep_set_neighbor_capacity(qnep_handle *h, int32_t cap_radial, int32_t cap_angular);

/*
 * qnep_compute: one force evaluation, enqueued on `cuda_stream`.
 *   pos_dev     [3][N] float64, component-major, Angstrom, any periodic image (wrapped inside)
 *   types_dev   [N] int32, 0..n_types-1
 *   box         [9] float64 HOST, rows = cell vectors a, b, c: any non-degenerate cell (PAPER.md :104; INVALID_ARG for zero
 *               volume); its perpendicular width along every cell vector must be >= r_c + skin (UNSUPPORTED otherwise);
 *               a PPPM mesh lives in the fractional coordinates of the cell
 *   want        QNEP_WANT_* flags; an output whose flag is clear may be NULL
 *   energy_dev  [1]    eV,   U^tot = U^NEP + U^ES (Eq. 4)
 *   forces_dev  [3][N] eV/A  (Eq. 11 + static electrostatic forces Eq. 15, 18 / 37)
 *   virial_dev  [9]    eV,   W_ab row-major, W = sum_i sum_j r_ij (x) F_ji + W^k,static (Eq. 12, 22) = -dU/d(strain)
 *   charges_dev [N]    e,    neutralised, unscaled q_i (Eq. 33)
 *   bec_dev     [9][N] e,    Z_i,ab at [(3a+b)][i] (Eq. 28), or NULL
 * Errors: INVALID_ARG, UNSUPPORTED, CUDA, OOM; NEIGHBOR_OVERFLOW / SKIN_VIOLATED / INVALID_ARG (a species index
 *         outside 0..n_types-1, detected on the device) of the PREVIOUS call.
 */
int qnep_compute(qnep_handle *h, int64_t n_atoms, const double *pos_dev, const int32_t *types_dev,
                 const double box[9], uint32_t want, double *energy_dev, double *forces_dev,
                 double *virial_dev, double *charges_dev, double *bec_dev, void *cuda_stream);

/*
 * qnep_compute_atom_virial: qnep_compute with the per-atom virial as an additional output:
 *   W_i = sum_j r_ij (x) F_ji                      for all partial forces: descriptor part (Eq. 14), dynamic-charge parts
 *                                                  (Eq. 16, 19 / 38, 23, folded) and the real-space static part (Eq. 15)
 *                                                  -- PAPER.md :130-132 Eq. 12, :149;
 *       + W_i^{k,static}                           Ewald: Re[ sum_k G q_i e^{ik.r_i} S(k) B ] / (4 pi eps0), PAPER.md
 *                                                  :179-185 Eq. 20-21 (real part: DESIGN.md reading G4);
 *                                                  PPPM: q_i / (4 pi eps0) sum_s W(r_i - r_s) F^-1[S G^opt B]_s,
 *                                                  :297-302 Eq. 39, six more inverse transforms.
 *   atom_virial_dev [9][N] float64 DEVICE, component-major, entry (3 a + b) * N + i = W_{i,ab}, eV; owned by the caller.
 *   sum_i W_i equals virial_dev up to rounding (Eq. 22).  `want` selects the other outputs as in qnep_compute
 *   (QNEP_WANT_BEC is not available here); forces are always evaluated.  Errors as qnep_compute.
 */
int qnep_compute_atom_virial(qnep_handle *h, int64_t n_atoms, const double *pos_dev, const int32_t *types_dev,
                             const double box[9], uint32_t want, double *energy_dev, double *forces_dev,
                             double *virial_dev, double *charges_dev, double *atom_virial_dev, void *cuda_stream);

/*
 * qnep_compute_host: the same evaluation with HOST buffers: copies positions (and, on calls that may rebuild the
 * neighbour list, the species: between builds the species of the last build apply, as in qnep_compute) to the device,
 * runs qnep_compute, copies the requested outputs back (the charges on a second stream while the evaluation goes on)
 * and synchronises the stream; device-side errors of THIS call are reported.  Layouts as above.
 */
int qnep_compute_host(qnep_handle *h, int64_t n_atoms, const double *pos_host, const int32_t *types_host,
                      const double box[9], uint32_t want, double *energy_host, double *forces_host,
                      double *virial_host, double *charges_host, double *bec_host, void *cuda_stream);

/*
 * qnep_md_run: n_steps of velocity-Verlet (kick-drift-kick) around qnep_compute, all on the device.
 *   pos_dev, vel_dev [3][N] float64, updated in place; mass_host[n_types] in amu;
 *   dt in natural units (Angstrom * sqrt(amu/eV); 1 fs = 1/10.180505);
 *   energy_dev[2]: potential and kinetic energy after the last step.
 * The first call computes the initial forces; forces are kept in the handle between calls, so consecutive calls
 * continue one trajectory (call qnep_md_reset before starting another one from different positions).
 * The neighbour policy set by qnep_set_neighbor_policy applies.  Synchronises at the end and reports
 * device-side errors (SKIN_VIOLATED, NEIGHBOR_OVERFLOW) of the run.
 */
int qnep_md_run(qnep_handle *h, int64_t n_atoms, double *pos_dev, double *vel_dev, const int32_t *types_dev,
                const double box[9], const double *mass_host, double dt, int32_t n_steps,
                double *energy_dev, void *cuda_stream);

/*
 * Outputs of the evaluations inside qnep_md_run.  By default a step evaluates energy and forces only (all an NVE run
 * needs).  With want = QNEP_WANT_VIRIAL and / or QNEP_WANT_CHARGES every step also evaluates the total virial / writes
 * the charges: virial_dev [9] and charges_dev [N] (DEVICE, owned by the caller, must stay valid for the following
 * qnep_md_run calls) hold the values of the LAST step when qnep_md_run returns.  want = 0 restores the default.
 * Errors: INVALID_ARG (a requested output pointer is null, or a flag other than VIRIAL / CHARGES).
 */
int qnep_md_set_outputs(qnep_handle *h, uint32_t want, double *virial_dev, double *charges_dev);

/*
 * Tell the handle that the caller changed positions or velocities behind qnep_md_run's back (a restart from a stored
 * state): the forces kept from the previous call are dropped and the next evaluation rebuilds the neighbour list.
 */
int qnep_md_reset(qnep_handle *h);

/*
 * CUDA graphs inside qnep_md_run: a step is ~25 kernel launches, which bounds small systems (a 3000-atom step is
 * ~0.1 ms of GPU work), so the step is captured once per kind (lists reused / rebuild) and replayed.
 * mode 0: never; 1 (default): when n_atoms <= 100000; 2: always.  Replayed steps carry no per-stage events
 * (qnep_profile_sum counts no evaluations for them).
 */
int qnep_set_md_graphs(qnep_handle *h, int32_t mode);

/*
 * Choice of the PPPM charge-assignment kernel (Eq. 35).  mode 0 (default): the shared-memory sweep kernel
 * when n_atoms >= 20000, the mesh has at least 1024 (y, z) columns of 8 x 8 points (256 x 256) and skin / 2 <= mesh
 * spacing, else one thread per atom; 1: always one thread per atom;
 * 2: the sweep kernel whenever skin / 2 <= mesh spacing (small systems too: used by the parity tests).  Both give the
 * same mesh up to the order of fp32 additions.  Errors: INVALID_ARG.
 */
int qnep_set_pppm_kernels(qnep_handle *h, int32_t mode);

/*
 * Kernel of the batched network contraction (the one stage where the north_star allows tensor cores).
 *   mode 2 (default for the 25-descriptor model with n_neurons <= 128): 5th-generation tensor cores, tcgen05.mma kind::tf32
 *           with accumulators and A operands in tensor memory and the 3xTF32 split (three products per term), which keeps
 *           FP32-level accuracy: site energies agree with mode 0 to ~3e-7 eV and the stated tolerances hold
 *           (tests/test_gpu_parity.py::test_nn_tensor_core_kernel).  0.201 ms on config 4.
 *   mode 1: warp-level mma.sync m16n8k8 TF32, same split (0.338 ms: the legacy path peaks at 277 TFLOP/s TF32 on B200).
 *   mode 0: packed FP32 FMAs, two atoms per thread (0.310 ms); the default when the 4-/5-body terms are on (one atom per
 *           thread, scalar) or n_neurons > 128.
 * Errors: INVALID_ARG, UNSUPPORTED (modes 1, 2 with the 4-/5-body terms on; mode 2 with n_neurons > 128; mode 1 when the weight
 *         tables of all species, n_types x (2 x 36 + 3) x n_neurons floats, exceed 200 KB of shared memory).
 */
int qnep_set_nn_kernel(qnep_handle *h, int32_t mode);

/*
 * Optional ZBL core repulsion (the paper defers to the NEP papers for it, PAPER.md :39; DESIGN.md
 * reading Z1).  enabled != 0 adds to every pair closer than r_outer the universal Ziegler-Biersack-Littmark potential
 *     U(r) = K Z_i Z_j / r * phi(r / a) * f_sw(r),   a = 0.46850 / (Z_i^0.23 + Z_j^0.23) Angstrom,
 *     phi(x) = 0.18175 e^{-3.19980 x} + 0.50986 e^{-0.94229 x} + 0.28022 e^{-0.40290 x} + 0.02817 e^{-0.20162 x},
 *     f_sw = 1 below r_inner, 1/2 [1 + cos(pi (r - r_inner) / (r_outer - r_inner))] up to r_outer, 0 beyond,
 * as a site energy 1/2 sum_j U(r_ij) per atom: it enters energy, forces, virial and per-atom virial; charges and
 * Born effective charges do not depend on it.  z_host [n_types] (HOST): atomic numbers, read during the call.
 * The term is evaluated on the angular pair list, hence r_outer <= rc_a.  enabled == 0 switches it off (other arguments
 * ignored).  Errors: INVALID_ARG (radii, atomic numbers), UNSUPPORTED (r_outer > rc_a).
 */
int qnep_set_zbl(qnep_handle *h, int32_t enabled, double r_inner, double r_outer, const double *z_host);

/* Synchronise the stream of the last call and report its device-side error state (OK, NEIGHBOR_OVERFLOW, SKIN_VIOLATED, CUDA). */
int qnep_check(qnep_handle *h);

/* CUDA-event times in milliseconds of the last qnep_compute, ms[QNEP_T_*]; n = number of entries to write. Synchronises. */
int qnep_get_timings(qnep_handle *h, float *ms_per_stage_host, int32_t n);

/*
 * Accumulated stage times: qnep_profile_reset() starts a window; qnep_profile_sum() synchronises and adds up the
 * CUDA-event stage times (ms[QNEP_T_*], as qnep_get_timings) of every evaluation since the reset, including those run
 * inside qnep_md_run (at most the 512 most recent); *n_evals = number of evaluations summed.  QNEP_T_FORCE_ANGULAR
 * brackets exactly one kernel launch per evaluation (the angular partial-force kernel).
 */
int qnep_profile_reset(qnep_handle *h);
int qnep_profile_sum(qnep_handle *h, float *ms_sum_host, int32_t n, int64_t *n_evals_host);

/* number of kernels launched by this handle since creation (bench.py's gpu_launches claim) */
int64_t qnep_kernel_launches(const qnep_handle *h);

/*
 * Response of the ions to a homogeneous external electric field and ionic polarization current (PAPER.md II.D,
 * Eq. 29-30, :229-237), from the Born effective charges Z written by qnep_compute (QNEP_WANT_BEC):
 *     F^ext_{i,b} = sum_a E_a Z_{i,ab}            (Eq. 29)        -> fext_dev [3][N], eV/A for E in V/A
 *     Pdot_a      = sum_i sum_b Z_{i,ab} v_{i,b}  (Eq. 30)        -> pdot_dev [3], e A / (time unit of v)
 * bec_dev : DEVICE, [9][N] component-major, entry (3 a + b) * N + i = Z_{i,ab} (a: polarization component,
 *           b: displacement component), the layout qnep_compute writes; owned by the caller.
 * efield  : HOST, 3 doubles, or NULL to skip Eq. 29 (fext_dev is then ignored).
 * vel_dev : DEVICE, [3][N] component-major, or NULL to skip Eq. 30 (pdot_dev is then ignored).
 * Enqueued on `cuda_stream`, no synchronisation.  Returns QNEP_ERR_INVALID_ARG for a null handle / bec pointer,
 * n_atoms <= 0, or a requested output whose pointer is null.
 */
int qnep_response(qnep_handle *h, int64_t n_atoms, const double *bec_dev, const double *efield_host,
                  const double *vel_dev, double *fext_dev, double *pdot_dev, void *cuda_stream);

/*
 * Neighbour statistics of the last call (synchronises): out[0], out[1] = max / mean length of the skin list
 * (r < rc_r + skin at build time); out[2], out[3] = max / mean number of radial neighbours inside rc_r;
 * out[4], out[5] = max / mean number of angular neighbours inside rc_a (the exact per-step lists).
 */
int qnep_neighbor_stats(qnep_handle *h, double out_host[6]);

/*
 * FP32 FMA throughput of the current device in TFLOP/s: a dependent-free FFMA loop on every SM, best of 4 launches,
 * CUDA-event timed on `cuda_stream`.  bench.py reports it beside the nominal FP32 peak.  Synchronises.
 */
int qnep_fma_peak(double *tflops_host, void *cuda_stream);

/*
 * Copy a per-stage intermediate of the last qnep_compute into a caller-owned DEVICE float64 buffer
 * (original atom order), for the per-stage parity tests.  `which` is a QNEP_DBG_* value; `n` is the
 * number of float64 elements `dst_dev` can hold.  Errors: INVALID_ARG.
 */
int qnep_debug_copy(qnep_handle *h, int32_t which, double *dst_dev, int64_t n);

/*
 * qnep_neutralise_noalloc: Eq. 33 (PAPER.md :255-262; reading G3) on its own, for callers that are not allowed to
 * allocate device memory:
 *     charges_i = q_raw_i + (q_total - sum_j q_raw_j) / n_atoms.
 * Everything else in this header sizes a workspace with cudaMalloc (qnep_create, and again when the atom count or the mesh
 * grows).  Some callers cannot do that: a plug-in of an MD engine or inference server whose own pool already holds the rest
 * of the GPU (a raw cudaMalloc from a library then fails, or takes memory the application had counted on); code in a
 * section that must not stall the device (cudaMalloc / cudaFree may synchronise the whole context and so every other
 * stream); code that must fix its memory footprint before the first step.  This entry point needs no handle and calls
 * neither cudaMalloc nor cudaFree nor any library routine that allocates: the one piece of scratch it needs, the partial
 * sums of q_raw, sits in an array compiled into the library (32 KiB, present on every GPU that loads the library until the
 * process ends).
 *   n_atoms      1 .. QNEP_NOALLOC_MAX_ATOMS; more is refused with QNEP_ERR_UNSUPPORTED and nothing is launched
 *   q_raw_dev    [n_atoms] float64 DEVICE, the network's charge outputs before Eq. 33 (what QNEP_DBG_Q_RAW returns)
 *   q_total      target total charge Q
 *   charges_dev  [n_atoms] float64 DEVICE, owned by the caller; may be the same buffer as q_raw_dev
 *   err_host     optional HOST buffer of err_len bytes that receives a message when the call fails (NULL: no message)
 * Two kernels are enqueued on `cuda_stream` (on the current device); the call does not synchronise.  The result does not
 * depend on the launch: every atom gets the same shift, summed in a fixed order.
 * First call on a device: looks up the device address of the built-in array (cudaGetSymbolAddress) and loads the two
 * kernels, once per device, with that device current.  Make that first call during start-up, outside any stream capture.
 * Shared state: all calls on one device use the same array, and it keeps the last call's contents.  Each call overwrites
 * the slots it reads before reading them, so nothing needs clearing between calls -- but calls whose kernels overlap on the
 * GPU (two streams without an event between them, two host threads) corrupt each other's sums: order them.
 * Errors: INVALID_ARG (null pointer, n_atoms <= 0), UNSUPPORTED (n_atoms above the maximum, device ordinal >= 64), CUDA.
 */
#define QNEP_NOALLOC_MAX_ATOMS 4194304 /* 4096 partial sums of 1024 atoms each */
int qnep_neutralise_noalloc(int64_t n_atoms, const double *q_raw_dev, double q_total, double *charges_dev,
                            void *cuda_stream, char *err_host, size_t err_len);

void qnep_destroy(qnep_handle *h);

/* Message of the last error on this handle (or of the last failed qnep_create if h == NULL); valid until the next call. */
const char *qnep_last_error(const qnep_handle *h);

#ifdef __cplusplus
}
#endif
#endif /* QNEP_H */
