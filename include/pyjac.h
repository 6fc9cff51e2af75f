/* pyjac.h -- C ABI of pyjac-b200: batched chemical-kinetic source terms and analytical Jacobians
 * (sparse CSR/CSC and dense) on one NVIDIA B200 (sm_100a), after pyJac v2, arXiv:1809.01029.
 *
 * Citations "PAPER.md Lnnn" refer to the paper text; "DESIGN.md Rn" to the readings listed there
 * for everything the paper defers to its (unavailable) supplement.
 *
 * State vector (Eq. 1):  phi = [T, E, n_1 .. n_{Ns-1}],  E = V (CONP) or P (CONV).
 * The other thermodynamic variable is the per-state PARAMETER: P for CONP, V for CONV.
 * n_var = Ns + 1.  The last species' concentration follows from the ideal-gas law and its rate from
 * mass conservation.
 * Source terms f = dphi/dt: PAPER.md Eqs. 2-8 (L128-164).  Jacobian J(i,j) = d f_i / d phi_j
 * (Eq. 9), 0-based: index 0 = T, 1 = E, 2+k = n_{k+1}.
 *
 * Units: T [K], P [Pa], V [m^3], n [kmol], concentrations [kmol/m^3], W [kg/kmol],
 * R = 8314.46261815324 J/(kmol K), P_atm = 101325 Pa.  Rate parameters in SI kmol-m^3-s, Ta = Ea/R [K].
 *
 * LAYOUT of every per-state device array (phi, dphi, sparse values, dense Jacobian):
 * element e (0 <= e < n_e) of state s (0 <= s < n_states) lives at
 *        (s / tile) * (n_e * tile)  +  e * tile  +  (s % tile)
 * with n_e = n_var (phi, dphi), nnz (sparse values), n_var^2 (dense; e = r*n_var + c for order 'C',
 * c*n_var + r for order 'F').  tile == ld is the pure structure-of-arrays / state-fastest layout (the
 * paper's "F" order); a small power-of-two tile is the paper's chunked "vectorised"
 * order (Fig. 3); tile == 1 is the state-major "C" order.
 * Constraints: ld >= n_states, ld % tile == 0, tile >= 1; tile is a power of two or tile == ld.
 * d_param is a plain [ld] array.  Base pointers must be 16-byte aligned.  Slots of states
 * s >= n_states are never read or written.
 *
 * OWNERSHIP: desc arrays are caller-owned HOST memory, copied by pyjac_mech_create.  The handle owns
 * its host and device tables.  State and output buffers are caller-owned DEVICE memory on the
 * handle's device.  The compute calls enqueue work on `stream` (a cudaStream_t passed as void*,
 * NULL = default stream) and return without synchronising; they allocate nothing and copy nothing
 * between host and device.  The *_host convenience calls take HOST buffers and do the copies
 * themselves (synchronous).
 *
 * ERRORS: every int-returning call returns PYJAC_OK or a nonzero status; pyjac_last_error() gives a
 * thread-local message.  State VALUES are not validated on the device (garbage in, NaN out).
 */
#ifndef PYJAC_H
#define PYJAC_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pyjac_mech pyjac_mech; /* opaque */

enum { PYJAC_OK = 0, PYJAC_EINVAL = 1, PYJAC_EMECH = 2, PYJAC_ECUDA = 3, PYJAC_ENOMEM = 4 };
enum { PYJAC_CONP = 0, PYJAC_CONV = 1 };                 /* mode */
enum { PYJAC_CSR = 0, PYJAC_CSC = 1 };                   /* sparse format */
enum { PYJAC_ELEMENTARY = 0, PYJAC_THIRD_BODY = 1, PYJAC_FALLOFF_LINDEMANN = 2, PYJAC_FALLOFF_TROE = 3,
       PYJAC_FALLOFF_SRI = 4, PYJAC_PLOG = 5, PYJAC_CHEBYSHEV = 6 };   /* reaction type */

/* Mechanism description ("all modern reaction types"; rate laws: DESIGN.md R2).
 * All pointers are HOST memory.  Ragged lists use CSR-style pointer arrays of length Nr+1. */
typedef struct {
  int32_t n_species, n_reactions;
  const double *mol_weight;                          /* [Ns] W_k, > 0                                  */
  const double *nasa_tmid, *nasa_lo, *nasa_hi;       /* [Ns], [Ns*7], [Ns*7]: a0..a6; low iff T<=tmid  */
  const int32_t *reac_ptr, *reac_species, *reac_nu;  /* reactants: <= 3 entries, integer nu' in 1..3   */
  const int32_t *prod_ptr, *prod_species, *prod_nu;  /* products, nu''                                 */
  const uint8_t *reversible;                         /* [Nr] 1: k_r = k_f / K_c, 0: k_r = 0            */
  const int32_t *type;                               /* [Nr] PYJAC_ELEMENTARY ..                       */
  const double *A, *beta, *Ta;                       /* [Nr] Arrhenius (k_inf for falloff), A > 0      */
  const int32_t *eff_ptr, *eff_species;              /* non-default third-body efficiencies, >= 0      */
  const double *eff_value;
  const int32_t *collider;                           /* [Nr] -1: mixture [M]; k: single collider (+X_k) */
  const double *low_A, *low_beta, *low_Ta;           /* [Nr] falloff low-pressure limit k_0            */
  const double *troe;                                /* [Nr*4] a, T3, T1, T2                           */
  const uint8_t *troe_has_T2;                        /* [Nr]                                           */
  const double *sri;                                 /* [Nr*5] a, b, c, d, e                           */
  const int32_t *plog_ptr;                           /* P-Log points, pressures strictly ascending [Pa] */
  const double *plog_P, *plog_A, *plog_beta, *plog_Ta;
  const int32_t *cheb_ptr, *cheb_nT, *cheb_nP;       /* Chebyshev: coefficient offset, grid sizes      */
  const double *cheb_Tmin, *cheb_Tmax, *cheb_Pmin, *cheb_Pmax; /* [Nr]                                 */
  const double *cheb_coef;                           /* row-major nT x nP, log10 of k in SI            */
  const uint8_t *chem_activated;                     /* [Nr] or NULL (= none).  1 on a falloff-type reaction:
                                                        chemically-activated bimolecular reaction (PAPER.md L143,
                                                        DESIGN.md R8): (A, beta, Ta) = k_inf and low_* = k_0 as for
                                                        falloff, P_r = k_0 [M] / k_inf, but k = k_0 F / (1 + P_r)   */
  const double *rev_A, *rev_beta, *rev_Ta;           /* [Nr] each, or all NULL (= none).  rev_A[i] > 0 on a reversible
                                                        reaction: explicit reverse rate constant k_r = A T^beta
                                                        exp(-Ta/T) instead of k_f / K_c (R9); not for P-Log
                                                        and Chebyshev reactions                                    */
} pyjac_mech_desc;

/* Step a0 (one-time, host): validate, sort reactions by type, pack device tables, build the exact
 * sparsity pattern in CSR and CSC and the static gather maps that replace the
 * paper's run-time index search.  Uploads the tables to `cuda_device`.
 * PYJAC_EMECH: Ns < 2, Nr < 1, index out of range, nu outside 1..3, more than 3 species per side,
 * A <= 0, W <= 0, tmid <= 0, negative efficiency, P-Log with < 2 points or non-ascending pressures,
 * empty Chebyshev grid or Tmin >= Tmax or Pmin >= Pmax, unknown type, chem_activated on a reaction that is not of a
 * falloff type, explicit reverse parameters on an irreversible, P-Log or Chebyshev reaction or rev_A < 0.  PYJAC_ECUDA: no such device.
 * cuda_device = -1 builds a HOST-ONLY handle (pyjac_mech_dims / pyjac_sparsity work; every compute
 * call fails with PYJAC_ECUDA) -- there is no CPU compute path.  The compute calls launch on the
 * caller's current device, which must be the handle's device. */
int pyjac_mech_create(const pyjac_mech_desc *desc, int cuda_device, pyjac_mech **out);

/* Same with flags.  PYJAC_APPROX_JACOBIAN selects the paper's "approximate" Jacobian: with the
 * third-body concentration written as [M] = C_tot + sum_k (alpha_k - 1) C_k, the derivatives of the rates of
 * progress and pressure-modification terms THROUGH THE LAST SPECIES' CONCENTRATION with respect to the other
 * species' moles are ignored (R6).  The dense rows caused by a reacting last species or by a non-default
 * efficiency of the last species disappear; pyjac_sparsity returns the sparser pattern; the T and E columns, the
 * source terms and everything else are unchanged.  For mechanisms whose last species is inert with default
 * efficiencies the two Jacobians are identical. */
enum { PYJAC_APPROX_JACOBIAN = 1, PYJAC_PAIR_KERNEL = 2 };
/* PYJAC_PAIR_KERNEL: evaluate the Jacobian with the pair-of-states kernel (a thread owns an item for
 * two states, the reactions are cut into blocks so that the per-reaction partials of one block fit on chip).  It is
 * chosen automatically for mechanisms whose partials do not fit in one SM's shared memory all at once; the flag forces it
 * for any mechanism (same results within the tolerances; tests and benchmarks). */
int pyjac_mech_create_ex(const pyjac_mech_desc *desc, int cuda_device, uint32_t flags, pyjac_mech **out);
void pyjac_mech_destroy(pyjac_mech *mech);

int pyjac_mech_dims(const pyjac_mech *mech, int32_t *ns, int32_t *nr, int32_t *nvar, int64_t *nnz);

/* Sparsity pattern of the n_var x n_var Jacobian (one pattern for CONP and CONV).  ptr has n_var+1
 * entries, idx has nnz entries, ascending inside each row (CSR) or column (CSC); CSC is the exact
 * transpose view of CSR.  The returned HOST pointers are owned by the handle.  Rule (R5):
 * rows and columns T, E dense; species block = union over reactions of
 * {k: nu_ki != 0} x {j: rate of i depends on C_j or on C_Ns, or alpha_ij != alpha_i,Ns}. */
int pyjac_sparsity(const pyjac_mech *mech, int fmt, const int32_t **ptr, const int32_t **idx);

/* Steps a1-a7: d_dphi = f(phi; param).  PAPER.md Eqs. 3-8. */
int pyjac_source_terms(const pyjac_mech *mech, int mode, int64_t n_states, int64_t ld, int64_t tile,
                       const double *d_phi, const double *d_param, double *d_dphi, void *stream);

/* Steps a1-a11: the nnz values of J per state, in the value order of `fmt`.  Every nonzero is
 * accumulated on chip and stored exactly once. */
int pyjac_jacobian_sparse(const pyjac_mech *mech, int mode, int fmt, int64_t n_states, int64_t ld,
                          int64_t tile, const double *d_phi, const double *d_param, double *d_vals,
                          void *stream);

/* pyjac_jacobian_sparse for callers that must not reach cudaMalloc'ed scratch or anything that allocates (code under
 * CUDA graph capture, tight serving loops, harnesses that forbid it): same arguments, same kernel, same results within
 * the parity tolerance, but the kernel's scratch -- the tile counter and the finished-CTA counter of the persistent
 * kernel -- lives in a file-scope static __device__ array of the library (256 bytes per GPU, held from the moment the
 * library is loaded until the process exits) instead of the handle's cudaMalloc'ed ring.  The call enqueues one
 * 16-byte cudaMemsetAsync (the counters must start at zero and keep the last call's contents) and one kernel on
 * `stream`; it calls no cudaMalloc, cudaFree, event or allocating routine and takes no lock.
 * LIMITS: n_states <= PYJAC_STATIC_MAX_STATES per call (PYJAC_EINVAL with a message otherwise: the static entry point
 * is meant for serving-size batches; larger batches are split by the caller or go through pyjac_jacobian_sparse).
 * EVERY call on a GPU shares the one scratch array: two calls that overlap on the GPU (different streams, different
 * handles, different host threads) RACE on the counters and skip or repeat tiles -- issue them on one stream, or order
 * them with events.  pyjac_jacobian_sparse has no such restriction. */
#define PYJAC_STATIC_MAX_STATES ((int64_t)1 << 22)
int pyjac_jacobian_sparse_static(const pyjac_mech *mech, int mode, int fmt, int64_t n_states, int64_t ld,
                                 int64_t tile, const double *d_phi, const double *d_param, double *d_vals,
                                 void *stream);

/* Steps a1-a11: all n_var^2 entries per state (structural zeros written as 0.0, each entry stored
 * exactly once; no memset pass).  order 'C': e = r*n_var + c, 'F': e = c*n_var + r. */
int pyjac_jacobian_dense(const pyjac_mech *mech, int mode, char order, int64_t n_states, int64_t ld,
                         int64_t tile, const double *d_phi, const double *d_param, double *d_J,
                         void *stream);

/* Conversions between the common mass / mole fractions and the state vector ("conversion to/from the
 * more-common mass/mole fractions and moles is straightforward"; Eq. 1).  d_frac holds ALL Ns fractions per
 * state in the library layout with n_e = Ns; d_T, d_P, d_V, d_param are plain [ld] arrays.
 *   from fractions:  X_k = (Y_k / W_k) / sum_j (Y_j / W_j) (mass fractions only);  n_k = X_k P V / (R T), k < Ns;
 *                    phi = [T, V | P, n_1 .. n_{Ns-1}], param = P | V.  The fractions need not be normalised for
 *                    kind = MASS (only ratios enter); for kind = MOLE they are used as given.
 *   from state:      X_k = n_k R T / (P V), k < Ns;  X_Ns = 1 - sum_{k<Ns} X_k (the last species' moles follow from the
 *                    ideal-gas law);  Y_k = X_k W_k / sum_j X_j W_j.
 * One elementwise kernel each on `stream`; no allocation, no synchronisation. */
enum { PYJAC_MOLE_FRACTION = 0, PYJAC_MASS_FRACTION = 1 };
int pyjac_state_from_fractions(const pyjac_mech *mech, int mode, int kind, int64_t n_states, int64_t ld, int64_t tile,
                               const double *d_T, const double *d_P, const double *d_V, const double *d_frac,
                               double *d_phi, double *d_param, void *stream);
int pyjac_fractions_from_state(const pyjac_mech *mech, int mode, int kind, int64_t n_states, int64_t ld, int64_t tile,
                               const double *d_phi, const double *d_param, double *d_frac, void *stream);

/* First-order forward finite-difference Jacobian: the paper's own comparison baseline (Fig. 12;
 * "implemented for comparison purposes only").  The paper gives no step rule; R7:
 *     xp_c = fl(phi_c + fma(rel_step, |phi_c|, abs_step)),  h_c = fl(xp_c - phi_c),
 *     J(i, c) = fl(fl(f_i(phi with phi_c := xp_c) - f_i(phi)) / h_c),
 * n_var + 1 source-term evaluations (steps a1-a7) per state, all inside one kernel.  fmt: PYJAC_CSR / PYJAC_CSC store
 * the nnz entries of the handle's pattern in that value order (entries outside the pattern are not formed); 'C' /
 * 'F' store all n_var^2 entries in that order.  rel_step, abs_step >= 0, not both 0 (PYJAC_EINVAL); a step that
 * rounds to h_c = 0 gives inf/NaN in that column.  Truncation error O(h): this is NOT the analytical Jacobian and is
 * only compared with an oracle doing the same arithmetic. */
int pyjac_jacobian_fd(const pyjac_mech *mech, int mode, int fmt, double rel_step, double abs_step, int64_t n_states,
                      int64_t ld, int64_t tile, const double *d_phi, const double *d_param, double *d_out, void *stream);

/* End-to-end convenience call on HOST buffers (same layouts): copy in, run, copy out, synchronise -- chunks of <= 8192
 * states double-buffered over two streams, so that with PINNED host buffers the copies overlap the kernels.  The
 * device staging buffers and the two streams belong to the handle: they are created by the first call (and grown if a
 * later call needs more) and freed by pyjac_mech_destroy, so repeated calls allocate nothing.  One pyjac_eval_host call
 * per handle at a time (calls from several threads serialise).  what: 0 = source terms, 1 = sparse Jacobian (fmt),
 * 2 = dense Jacobian (fmt = 'C' or 'F').  h_out must hold n_e * ld doubles. */
int pyjac_eval_host(const pyjac_mech *mech, int what, int mode, int fmt, int64_t n_states, int64_t ld,
                    int64_t tile, const double *h_phi, const double *h_param, double *h_out);

/* Launch geometry the library chooses for a call with these n_states and tile (the ONE launch policy; bench.py and
 * the tests ask here): states per CTA, threads per CTA, dynamic shared memory bytes.  what as in pyjac_eval_host;
 * 3 = finite-difference Jacobian (states_per_cta is then the number of perturbed columns one CTA evaluates per pass
 * over its single state).  n_states <= 0 means "a large batch", tile <= 0 "any layout".  States per CTA: the largest
 * power of two whose intermediates fit in shared memory, that does not exceed `tile`, and that still leaves two tiles
 * per SM of the handle's device. */
int pyjac_launch_info(const pyjac_mech *mech, int what, int64_t n_states, int64_t tile, int32_t *states_per_cta,
                      int32_t *threads, int64_t *smem_bytes);

/* Shape of the Jacobian kernel's gather plan, for reporting: info[0] = H (reaction blocks per
 * state pair), [1] = value slots of the largest block, [2] = partial-sum slots, [3] = gather entries, [4] = stored
 * entries (with ELL padding), [5] = groups, [6] = piece slots, [7] = lists cut into more than one piece. */
int pyjac_plan_info(const pyjac_mech *mech, int64_t info[8]);

/* Machine peaks measured on `cuda_device` (the denominators of the rooflines bench.py reports; SURVEY.md section
 * 8d asks for a measured DFMA rate and a measured write-only stream instead of datasheet figures).  Each figure is
 * timed with CUDA events around `reps` back-to-back launches after one warm-up launch; the call allocates its own
 * scratch (up to 8 GiB for the copy) and synchronises.  *value: DFMA per second (PYJAC_PEAK_DFMA: 8 independent
 * chains per thread, 2048 threads per SM) or bytes per second (the others: 4 GiB streams with 16-byte accesses;
 * PYJAC_PEAK_L2_READ: every CTA sweeps one L2-resident 32 MiB window with ld.global.cg; PYJAC_PEAK_LDS:
 * conflict-free 16-byte shared-memory loads). */
enum { PYJAC_PEAK_DFMA = 0, PYJAC_PEAK_HBM_WRITE = 1, PYJAC_PEAK_HBM_READ = 2, PYJAC_PEAK_HBM_COPY = 3,
       PYJAC_PEAK_L2_READ = 4, PYJAC_PEAK_LDS = 5 };
int pyjac_measure_peak(int kind, int cuda_device, int reps, double *value);

const char *pyjac_last_error(void); /* thread-local, never NULL */

#ifdef __cplusplus
}
#endif
#endif /* PYJAC_H */
