/* pyjac_b200.h -- C ABI of the B200-native batched chemical-kinetics source term and analytical
 * Jacobian (the method of arxiv 1605.03262, "pyJac", evaluated from tables instead of generated code).
 *
 * Citations are PAPER.md:<line> plus the equation they fall in.  Units: SI with kmol
 * (J, kmol, m^3, K, Pa); R = 8314.46261815324 J kmol^-1 K^-1, p_atm = 101325 Pa.
 *
 * For every thermochemical state (T, P, Y_1..Y_Nsp) the library evaluates, on the GPU only
 * (sm_100a kernels; there is no CPU fallback and every call fails with PYJAC_ECUDA if no device
 * is usable):
 *   - NASA-7 thermodynamics                                   PAPER.md:118-134 Eqs. 9-13
 *   - forward / reverse rates of progress R_f, R_r            PAPER.md:150-155 Eqs. 17-19
 *     with Arrhenius, PLOG and Chebyshev rate coefficients    PAPER.md:166 Eq. 21, :251-259
 *                                                             Eqs. 37-39, :264-278 Eqs. 40-43
 *     and k_r = k_f / K_c or explicit reverse parameters      PAPER.md:181-199 Eqs. 23-27
 *   - the pressure modification c_i (third body, Lindemann / Troe / SRI falloff,
 *     chemically activated)                                   PAPER.md:159 Eq. 20, :206-245 Eqs. 28-36
 *   - species production rates and the constant-pressure source term dPhi/dt
 *                                                             PAPER.md:140 Eq. 14, :102-108 Eqs. 6-8
 *   - the dense analytical Jacobian d(dPhi/dt)/dPhi           PAPER.md:288-570 Eqs. 44-113,
 *     in the reaction-wise evaluation order of Section 4      PAPER.md:609-744 Alg. 2, Eqs. 115-130
 *
 * Bench / test helpers (table statistics, machine-peak probes) are NOT part of this interface:
 * they live in include/pyjac_b200_tools.h and a library of their own.  The library reads no
 * environment variable; everything it does follows from the call arguments.
 *
 * Conventions
 *   - Every function returns 0 (PYJAC_OK) or a negative error code; nothing throws or exits.
 *   - `pyjac_mech_desc` holds HOST pointers; the library copies what it needs during
 *     pyjac_mech_create and never keeps a caller pointer.
 *   - Array arguments of the pyjac_eval_* calls are DEVICE pointers on the handle's device, owned by
 *     the caller (never freed or retained).  The *_host variants take HOST pointers instead.
 *   - pyjac_eval_* enqueue on `stream` (a cudaStream_t passed as void*; NULL = the legacy default
 *     stream), allocate nothing and do not synchronise.  A handle is immutable after creation:
 *     evaluation is re-entrant and may be called from several host threads / streams at once.
 *   - Results do not depend on n, on how a batch is split, or on the stream: every sum is taken in
 *     an order fixed at pyjac_mech_create (bit-identical re-evaluation).
 *   - Inputs are not checked on the device.  The caller guarantees T > 0, P > 0, Y_k >= 0 and, for
 *     falloff / chemically-activated reactions, a non-zero third-body concentration [X]_i
 *     (PAPER.md:385 discusses the zero-concentration hazard; products that skip a factor are used
 *     instead of divisions by [X_j], so Y_k = 0 is allowed).
 *   - State layout: T[n] (K), P[n] (Pa), Y[s*ldy + k] for state s, species k = 0..Nsp-1, ldy >= Nsp.
 *     All Nsp mass fractions are supplied; Y_Nsp is used as given (it equals Eq. 2, PAPER.md:84,
 *     when sum_k Y_k = 1), derivatives are taken under the Eq. 2 constraint.
 */
#ifndef PYJAC_B200_H
#define PYJAC_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* error codes */
#define PYJAC_OK 0
#define PYJAC_EINVAL (-1) /* bad argument or inconsistent mechanism description */
#define PYJAC_ENOMEM (-2) /* host or device allocation failed */
#define PYJAC_ECUDA (-3)  /* CUDA runtime / launch error (no device, wrong architecture, ...) */
#define PYJAC_ELIMIT (-4) /* mechanism exceeds a table limit of this build (see pyjac_mech_create) */
#define PYJAC_ESCRATCH (-5) /* batch too large for the built-in scratch array (pyjac_eval_jacobian_fd_static) */

/* rxn_type: which case of Eq. 20 / which rate form applies */
enum {
    PYJAC_ELEMENTARY = 0,     /* c_i = 1, Arrhenius k_f (Eq. 21) */
    PYJAC_THIRD_BODY = 1,     /* c_i = [X]_i (Eqs. 28-30) */
    PYJAC_FALLOFF = 2,        /* c_i = P_r/(1+P_r) F, k_f = k_inf (Eqs. 31-36) */
    PYJAC_CHEM_ACTIVATED = 3, /* c_i = F/(1+P_r),     k_f = k_0 */
    PYJAC_PLOG = 4,           /* c_i = 1, k_f by Eqs. 37-39 */
    PYJAC_CHEBYSHEV = 5       /* c_i = 1, k_f by Eqs. 40-43 */
};
/* rev_type */
enum { PYJAC_IRREVERSIBLE = 0, PYJAC_REV_FROM_KC = 1 /* Eq. 23 */, PYJAC_REV_EXPLICIT = 2 };
/* falloff_form (Eq. 32) */
enum { PYJAC_LINDEMANN = 0, PYJAC_TROE = 1, PYJAC_SRI = 2 };

/* Kinetic model description.  All pointers are HOST pointers, read only during pyjac_mech_create.
 * Arrays sized [n_reactions][..] must be present for every reaction (entries of reactions they do
 * not apply to are ignored), except the CSR payload arrays, which may be NULL when empty. */
typedef struct pyjac_mech_desc {
    int32_t n_species;         /* N_sp >= 1; the LAST species is the one eliminated by Eq. 2 */
    int32_t n_reactions;       /* N_reac >= 0 */
    const double *mol_wt;      /* [N_sp] W_k, kg/kmol (Eq. 4) */
    const double *nasa_lo;     /* [N_sp][7] a_0..a_6 for T <= t_mid[k] (Eqs. 9-11) */
    const double *nasa_hi;     /* [N_sp][7] a_0..a_6 for T >  t_mid[k] */
    const double *t_mid;       /* [N_sp] */
    /* stoichiometry, CSR per reaction: nu'_ki (reactants) and nu''_ki (products), Eq. 15.
     * At most 3 entries per side, integer nu in 1..3, species distinct within a side. */
    const int32_t *reac_ptr;   /* [N_reac+1] */
    const int32_t *reac_spec;  /* species index 0..N_sp-1 */
    const int32_t *reac_nu;
    const int32_t *prod_ptr;   /* [N_reac+1] */
    const int32_t *prod_spec;
    const int32_t *prod_nu;
    const int32_t *rxn_type;   /* [N_reac] PYJAC_ELEMENTARY .. PYJAC_CHEBYSHEV */
    const int32_t *rev_type;   /* [N_reac] */
    const double *arr_hi;      /* [N_reac][3] (A, beta, T_a [K]) of Eq. 21; k_inf for FALLOFF and
                                  CHEM_ACTIVATED; unused for PLOG / CHEBYSHEV.  A > 0. */
    const double *arr_lo;      /* [N_reac][3] k_0 (FALLOFF, CHEM_ACTIVATED only) */
    const double *arr_rev;     /* [N_reac][3] explicit reverse parameters (REV_EXPLICIT only) */
    const int32_t *falloff_form; /* [N_reac] */
    const double *falloff_par; /* [N_reac][5] Troe: a, T***, T*, T**, has_T** (0/1) (Eq. 33);
                                  SRI: a, b, c, d, e (Eq. 36; d = 1, e = 0 when absent) */
    const int32_t *tb_species; /* [N_reac] m >= 0: [X]_i = [X_m] (Eq. 30); -1: mixture (Eq. 28) */
    const int32_t *eff_ptr;    /* [N_reac+1] CSR of third-body efficiencies alpha_ij != 1 (Eq. 28) */
    const int32_t *eff_spec;
    const double *eff_val;
    const int32_t *plog_ptr;   /* [N_reac+1] CSR of PLOG rows, >= 2 per PLOG reaction */
    const double *plog_p;      /* pressures in Pa, strictly ascending within a reaction */
    const double *plog_arr;    /* [][3] (A, beta, T_a) at each pressure (Eqs. 37-38) */
    const int32_t *cheb_ptr;   /* [N_reac+1] offsets into cheb_eta */
    const int32_t *cheb_nT;    /* [N_reac] N_T (Eq. 40) */
    const int32_t *cheb_nP;    /* [N_reac] N_p */
    const double *cheb_lim;    /* [N_reac][4] T_min, T_max, p_min, p_max (Eqs. 42-43) */
    const double *cheb_eta;    /* eta_ij, row-major in (i, j) (Eq. 40) */
} pyjac_mech_desc;

typedef struct pyjac_mech pyjac_mech; /* opaque, owned by the library */

/* Validates the description, sorts and packs it into device-resident SoA tables (precomputing
 * ln A, sum nu, the reaction-wise contribution lists of Algorithm 2) and
 * uploads them to CUDA device `device`.  The launch shape (states a CTA interleaves, threads per
 * CTA, CTAs per SM) is chosen from the size of the per-state tables.
 * Errors: PYJAC_EINVAL (NULL pointers, counts < 0, indices out of range, nu outside 1..3, more than
 * 3 species on a side, A <= 0, non-ascending PLOG pressures, T_min >= T_max, ...), PYJAC_ELIMIT
 * (more than 65534 species, 65535 reactions or 65535 per-state table entries, or per-state
 * tables that exceed the 227 KB of shared memory of one CTA), PYJAC_ENOMEM, PYJAC_ECUDA. */
int pyjac_mech_create(const pyjac_mech_desc *host_desc, int device, pyjac_mech **out);

/* Launch shape of the evaluation kernels; 0 in a field = let the library choose.  The kernels
 * evaluate `states_per_cta` states per CTA iteration, interleaved in shared memory (PAPER.md:857
 * names cache capacity as what limits its one-thread-per-state layout; here the per-state
 * reaction products stay in shared memory instead). */
typedef struct pyjac_launch_shape {
    int32_t states_per_cta; /* 1, 2, 3, 4 or 6 */
    int32_t threads;        /* per CTA: a multiple of 32, at least 64 and 32 * states_per_cta, at most 512 */
    int32_t ctas_per_sm;    /* resident CTAs the shared-memory footprint is sized for, 1..4 */
    int32_t list_cap;       /* longest list one lane sums in the per-species / per-column phase; longer
                               lists are shared by 2, 4, .. lanes and combined by warp shuffles */
    int32_t cell_cap;       /* 1..3: longest contribution list of a Jacobian entry summed while the
                               column is streamed out; longer lists are summed piecewise before */
    int32_t rows_per_lane;  /* 1 or 2 Jacobian rows per lane in the streaming phase (2 needs N_sp odd,
                               i.e. an even leading dimension; 16-byte stores) */
    int32_t p1_states;      /* states one work item of the reaction phase evaluates with the reaction's
                               constants held in registers: p + 16 g = p states per item of a group of plain
                               elementary reactions, g per item of a group with other rate forms (g = 0: p);
                               0: all states_per_cta for plain groups, one for the others */
    int32_t stage_tables;   /* 1: copy the gather tables to shared memory once per CTA (PYJAC_ELIMIT if they
                               do not fit this shape); 0: read them through L1 / L2 */
    int32_t layout;         /* 2: keep the per-reaction terms in allocation order in shared memory; 0 / 1: place
                               them so that the gathers meet few bank conflicts (same numbers either way) */
} pyjac_launch_shape;

/* As pyjac_mech_create with an explicit launch shape (tuning and tests; `shape` may be NULL).
 * Every shape evaluates the same numbers up to the order of a sum.  PYJAC_EINVAL for a value out
 * of range -- explicit values are never adjusted: too few threads for states_per_cta, rows_per_lane = 2
 * with an even N_sp or a negative field are errors -- PYJAC_ELIMIT if the shape does not fit the shared
 * memory of one SM. */
int pyjac_mech_create_shaped(const pyjac_mech_desc *host_desc, int device,
                             const pyjac_launch_shape *shape, pyjac_mech **out);

/* Why the last pyjac_mech_create / pyjac_mech_create_shaped call of THIS host thread failed: a static,
 * never-NULL sentence naming the rule that was broken ("nu outside 1..3", "PLOG pressures must ascend",
 * "threads per CTA must be ...", ...); "" after a call that succeeded. */
const char *pyjac_mech_create_error(void);

/* Frees the device tables.  NULL is a no-op returning PYJAC_OK. */
int pyjac_mech_destroy(pyjac_mech *mech);

/* Queries N_sp and N_reac (either output may be NULL). */
int pyjac_mech_sizes(const pyjac_mech *mech, int32_t *n_species, int32_t *n_reactions);

/* Rates of progress and production rates for n states.  Outputs (any may be NULL = skipped), all
 * state-major in the ORIGINAL reaction / species order:
 *   rf[n][N_reac], rr[n][N_reac]  R_f,i and R_r,i of Eqs. 18-19 (before c_i), kmol m^-3 s^-1 (times
 *                                  1/[X]_i for third-body and falloff forms)
 *   cmod[n][N_reac]                c_i of Eq. 20 (1 for elementary / PLOG / Chebyshev)
 *   wdot[n][N_sp]                  species production rates of Eq. 14, kmol m^-3 s^-1 */
int pyjac_eval_rates(const pyjac_mech *mech, int64_t n, const double *T, const double *P,
                     const double *Y, int64_t ldy, double *rf, double *rr, double *cmod,
                     double *wdot, void *stream);

/* Source term: dydt[n][N_sp+1] = { dT/dt (Eq. 7), dY_1/dt .. dY_Nsp/dt (Eq. 8) }, i.e. the paper's
 * f (Eq. 6) followed by the rate of the last ("placeholder") species. */
int pyjac_eval_dydt(const pyjac_mech *mech, int64_t n, const double *T, const double *P,
                    const double *Y, int64_t ldy, double *dydt, void *stream);

/* Analytical Jacobian: jac[n][(N_sp+1)^2], per state column-major with leading dimension
 * LD = N_sp+1, element (r, c) at r + c*LD; r, c = 0 <-> T; r, c = k <-> Y_k (k = 1..N_sp).
 * Rows/columns 0..N_sp-1 are exactly the paper's Jacobian J_{i,j} = d f_i / d Phi_j (Eqs. 44-49);
 * row N_sp is the placeholder row of PAPER.md:570 (d(dY_Nsp/dt)/dPhi_j, which the method computes
 * anyway for the energy row, Eq. 113); column N_sp is zero (Y_Nsp is not independent, Eq. 2). */
int pyjac_eval_jacobian(const pyjac_mech *mech, int64_t n, const double *T, const double *P,
                        const double *Y, int64_t ldy, double *jac, void *stream);

/* Jacobian-vector product without the matrix: jv[n][N_sp+1] = J v per state, J the matrix of
 * pyjac_eval_jacobian (rows 0..N_sp, the placeholder row included) and v[n][ldv] one vector per state
 * with entries 0..N_sp (entry N_sp multiplies the zero column and is not read); ldv >= N_sp+1.  This is
 * what a matrix-free implicit integrator consumes (the paper's motivation): the
 * (N_sp+1)^2 doubles per state never go to memory.  The column sum is taken per reaction first,
 *   (J v)_{k+1} = W_k sum_i nu_ki tau_i,  tau_i = sum_j s'_ij v_j / W_j + (U a_i + v_0 Theta_i) / rho,
 * with the per-reaction products of Section 4.1, so the cost is
 * that of the source term, O(N_reac), not O(N_sp^2).  Device pointers, asynchronous on `stream`. */
int pyjac_eval_jvp(const pyjac_mech *mech, int64_t n, const double *T, const double *P,
                   const double *Y, int64_t ldy, const double *v, int64_t ldv, double *jv,
                   void *stream);

/* Host-buffer variants: T, P, Y and the output are HOST pointers (pinned memory makes the copies
 * asynchronous; pageable memory works but serialises them).  The call copies the inputs to the
 * device, runs the same kernels as above in chunks of at most `chunk_states` states (<= 0: a
 * default whose output buffer is at most 512 MiB and a quarter of the device's free memory), copies
 * the result back with copies of one chunk overlapping the evaluation of the next, and returns after
 * the last byte has arrived.  The two device staging buffer pairs and the two streams are kept with
 * the handle and reused by later calls (grown when a call needs more): with the default chunk that is
 * up to ~1.1 GiB of device memory per handle, held until pyjac_mech_trim or pyjac_mech_destroy.  A
 * call whose explicit `chunk_states` needs a buffer above 512 MiB, and a second thread that calls
 * while the kept buffers are in use, stage through temporary buffers freed before the call returns. */
int pyjac_eval_jacobian_host(const pyjac_mech *mech, int64_t n, const double *T, const double *P,
                             const double *Y, int64_t ldy, double *jac, int64_t chunk_states);
int pyjac_eval_dydt_host(const pyjac_mech *mech, int64_t n, const double *T, const double *P,
                         const double *Y, int64_t ldy, double *dydt, int64_t chunk_states);

/* Frees the staging buffers the *_host calls left with the handle (no-op returning PYJAC_OK when there
 * are none or while a *_host call is using them).  The handle stays usable; the next *_host call
 * allocates again. */
int pyjac_mech_trim(pyjac_mech *mech);

/* First-order forward-difference Jacobian from the source term (the paper's own comparison: "a simple
 * first-order forward difference adapted from CVODE", Tables 4-5), in
 * the layout of pyjac_eval_jacobian.  With Phi = (T, Y_1 .. Y_{Nsp-1}), N = N_sp unknowns, f = dPhi/dt:
 *   w_j = 1 / (rtol |Phi_j| + atol),  D_j = max(sqrt(eps) |Phi_j|, sqrt(eps) / w_j),
 *   J(:, j) = (f(Phi + D_j e_j) - f(Phi)) / D_j
 * (CVODE's rule with its step-dependent floor 1000 |h| eps N |f| replaced by sqrt(eps): DESIGN.md C21),
 * a mass-fraction increment being taken from Y_Nsp (Eq. 2); column N_sp is zero.  rtol > 0 and atol > 0
 * (PYJAC_EINVAL otherwise: with atol = 0 an unknown that is exactly zero, as absent species are, would get
 * D_j = 0 and a column of 0/0).
 * All pointers are DEVICE pointers.  `work` is caller-owned scratch of `work_doubles` doubles; the
 * states are evaluated in chunks of work_doubles / pyjac_fd_workspace_doubles(mech, 1) states
 * (PYJAC_EINVAL if that is zero): 1 + N_sp source-term evaluations per state, 4 kernel launches
 * per chunk, asynchronous on `stream`, no allocation. */
int pyjac_eval_jacobian_fd(const pyjac_mech *mech, int64_t n, const double *T, const double *P,
                           const double *Y, int64_t ldy, double rtol, double atol, double *jac,
                           double *work, int64_t work_doubles, void *stream);

/* Doubles of scratch pyjac_eval_jacobian_fd needs to evaluate `chunk_states` states at once
 * (-1 for an invalid argument). */
int64_t pyjac_fd_workspace_doubles(const pyjac_mech *mech, int64_t chunk_states);

/* pyjac_eval_jacobian_fd for callers that cannot allocate device memory and so have no `work` buffer to
 * pass: a flow solver that gave the whole GPU to its own arena at start-up (any later cudaMalloc fails), an
 * integrator callback inside a time-step loop where cudaMalloc / cudaFree would stall every stream of the
 * device through their device-wide synchronisation, a plug-in whose host forbids driver allocations after
 * initialisation.  Same operation, arguments, layout and numbers (bit for bit) as pyjac_eval_jacobian_fd
 * (C21); the caller still owns T, P, Y and jac (DEVICE pointers).  The scratch is an
 * array compiled into the library: 4 Mi doubles = 32 MiB of device memory, which every GPU that loads the
 * library holds until the process exits whether or not this function is ever called.
 *   - Limit: all n states of a call must fit the array at once, n <= pyjac_fd_static_max_states(mech)
 *     (32 MiB / pyjac_fd_workspace_doubles(mech, 1) doubles: 712 states at 53 species, 166 at 111, 16 at 360).
 *     A larger n, or a mechanism of which not even one state fits, returns PYJAC_ESCRATCH and enqueues
 *     nothing; loop over sub-batches instead.  Other errors as pyjac_eval_jacobian_fd.
 *   - The function and everything under it call no cudaMalloc, cudaFree or other allocating routine.
 *   - The first call on each device looks the array's device address up (cudaGetSymbolAddress, with that
 *     device made current for the moment); this is host-side set-up, possibly a module load.  Make that
 *     first call early, before any stream capture is begun on the thread.  Later calls only enqueue the
 *     four kernels on `stream`.
 *   - There is ONE array per GPU, shared by every handle, stream and host thread.  Two calls whose kernels
 *     can overlap on the GPU (different streams without an ordering between them, or two host threads)
 *     race on it and produce garbage: order them on one stream or with events.  The array keeps whatever
 *     the last call wrote; this path never reads a scratch word before writing it in the same call, so no
 *     clearing is needed and stale contents cannot leak into a result. */
int pyjac_eval_jacobian_fd_static(const pyjac_mech *mech, int64_t n, const double *T, const double *P,
                                  const double *Y, int64_t ldy, double rtol, double atol, double *jac,
                                  void *stream);

/* Largest n pyjac_eval_jacobian_fd_static accepts for this mechanism (0 if one state does not fit the
 * 32 MiB array; -1 for an invalid handle). */
int64_t pyjac_fd_static_max_states(const pyjac_mech *mech);

/* Number of kernel launches this library has enqueued since it was loaded (all handles). */
int64_t pyjac_kernel_launches(void);

/* Launch configuration the Jacobian kernel uses for this mechanism (any output may be NULL):
 * threads per CTA, dynamic shared memory per CTA in bytes, resident CTAs per SM, grid size for n
 * states, states a CTA interleaves per iteration.  Reported by bench.py next to the roofline numbers. */
int pyjac_jacobian_launch_config(const pyjac_mech *mech, int64_t n, int32_t *threads,
                                 int32_t *smem_bytes, int32_t *ctas_per_sm, int32_t *grid,
                                 int32_t *states_per_cta);

/* Static, never-NULL description of an error code. */
const char *pyjac_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* PYJAC_B200_H */
