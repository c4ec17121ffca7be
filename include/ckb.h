/*
 * ckb.h -- C ABI of the batched chemical-kinetics integrator for B200 (sm_100a, FP64).
 *
 * The library advances N independent constant-pressure chemistry ODE systems
 *     y = {T, Y_1 .. Y_K}
 * over one global flow step dt by adaptive explicit integration, statelessly ("take as input
 * initial conditions and a global time step, performing internal sub-stepping as necessary"):
 *     method 0 : RKCK, 5th-order Runge-Kutta-Cash-Karp with embedded 4th-order error estimate
 *                (Eq. 7-17, Table 1)
 *     method 1 : RKC, stabilised 2nd-order Runge-Kutta-Chebyshev (Eq. 18-39) with the
 *                nonlinear power-method spectral-radius estimate and per-step stage count
 * Source term f(y): Eq. 2-6: Arrhenius rate coefficients (Eq. 5), third-body concentrations
 * (P:80), mass-action rates of progress (Eq. 4), net production rates (Eq. 3), NASA-polynomial cp / h
 * for the temperature equation (Eq. 6).  Readings of the paper where it is silent: DESIGN.md section 4.
 *
 * Every step of that path runs in hand-written CUDA kernels; there is no CPU fallback.  All entry
 * points return CKB_OK (0) or a negative error code; ckb_strerror() gives the text.
 *
 * Units (cgs): mol, cm, s, K; activation energy in cal/mol; molecular weight in g/mol; pressure in
 * dyn/cm^2.
 */
#ifndef CKB_H_
#define CKB_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CKB_OK 0
#define CKB_EINVAL (-1)       /* null pointer, bad shape, inconsistent CSR, index out of range       */
#define CKB_ENOMEM (-2)       /* host or device allocation failed                                    */
#define CKB_ECUDA (-3)        /* a CUDA runtime call failed; text via ckb_last_cuda_error()          */
#define CKB_EUNSUPPORTED (-4) /* mechanism outside the packed format's limits (see ckb_mech_load)    */
#define CKB_ECAPACITY (-5)    /* batch larger than the size reserved for the handle (ckb_mech_reserve) */

#define CKB_METHOD_RKCK 0
#define CKB_METHOD_RKC 1

/* variant: how ODE systems are mapped onto lanes */
#define CKB_VARIANT_AUTO 0    /* K+1 > 16: warp.  K+1 <= 16: warp for small N, 4 lanes from N = 12288 (RKC:
                                 24576), thread from N = 131072 (RKC: 196608); after ckb_mech_specialize
                                 thread from N = 49152 (RKC: 98304)                                     */
#define CKB_VARIANT_THREAD 1  /* one thread integrates one system (the paper's mapping)        */
#define CKB_VARIANT_WARP 2    /* one warp integrates one system; species and reactions over lanes     */
#define CKB_VARIANT_SUB8 3    /* 8 lanes per system (4 systems per warp)                              */
#define CKB_VARIANT_SUB16 4   /* 16 lanes per system (2 systems per warp)                             */
#define CKB_VARIANT_SUB2 5    /* 2 lanes per system (K+1 <= 16)                                        */
#define CKB_VARIANT_SUB4 6    /* 4 lanes per system (K+1 <= 16)                                        */

/* per-system status codes written to status[] */
#define CKB_ST_OK 0
#define CKB_ST_MAXSTEPS 1     /* more than 10^6 step attempts                                         */
#define CKB_ST_UNDERFLOW 2    /* step size fell below 10 u max(|t|,|t+dt|)                            */
#define CKB_ST_NONFINITE 3    /* as 2, after a non-finite trial state                                 */
#define CKB_ST_SIGMA 4        /* RKC: power method did not converge in 50 iterations (result kept)    */

/*
 * Mechanism description: plain HOST arrays, caller-owned, copied during ckb_mech_load.
 * Irreversible reactions only (every reversible reaction is entered as two irreversible ones).
 */
typedef struct {
  int32_t n_species;           /* K, 1..254                                                         */
  int32_t n_reactions;         /* R irreversible reactions                                          */
  const double *mol_weight;    /* [K]    W_k, g/mol                                                 */
  const double *nasa;          /* [K][7] a1..a7 of one temperature range (a7 unused on this path)   */
  const double *arr_A;         /* [R]    pre-exponential A_j (Eq. 5), cgs, > 0                      */
  const double *arr_beta;      /* [R]    temperature exponent                                       */
  const double *arr_E;         /* [R]    activation energy, cal/mol                                 */
  const int32_t *reac_ptr;     /* [R+1]  CSR over reactant entries                                  */
  const int32_t *reac_species; /* [nnz]  species index 0..K-1                                       */
  const int32_t *reac_nu;      /* [nnz]  nu'_kj  >= 1 (integer reaction order = stoichiometry)      */
  const int32_t *prod_ptr;     /* [R+1]  CSR over product entries                                   */
  const int32_t *prod_species; /* [nnz]                                                             */
  const int32_t *prod_nu;      /* [nnz]  nu''_kj >= 1                                               */
  int32_t n_third_body;        /* R3 reactions that carry a third body +M                    */
  const int32_t *tb_reaction;  /* [R3]   reaction index                                             */
  const int32_t *tb_ptr;       /* [R3+1] CSR over listed (non-unity) efficiencies                   */
  const int32_t *tb_species;   /* [nnz]                                                             */
  const double *tb_eff;        /* [nnz]  alpha_jk; every species not listed has alpha = 1           */
} ckb_mech_desc;

typedef struct ckb_mech ckb_mech; /* opaque; owns the packed tables in device memory */

/*
 * ckb_mech_load: validate `d`, pack it into the device tables of DESIGN.md section 6.1 (forward /
 * reverse reactions over the same species are fused into one slot; species-major gather lists for
 * Eq. 3; third-body efficiency sets), upload them to the current CUDA device, and return a handle in
 * *out (library-owned; release with ckb_mech_free).  Synchronous.
 * It also allocates everything ckb_integrate will ever need for this handle: the work-queue order scratch for
 * batches of up to CKB_DEFAULT_MAX_BATCH systems (12 bytes per system; ckb_mech_reserve changes the size) and, for
 * mechanisms with K+1 > 16, the stage-vector workspace of the thread-per-ODE variant (64 (K+1) bytes per resident
 * lane: 131 MB for K = 53 on a 148-SM device).
 * Limits (CKB_EUNSUPPORTED): K <= 254; at most 3 molecules (sum of nu) on either side of a reaction; at most 65000
 * distinct third-body efficiency sets; per mapping, the shared-memory region of a system is addressed with 16-bit
 * byte offsets: (K+1 + sets + fused reaction slots rounded up to the lanes per system + 16) * 8 <= 65535 for the
 * lane-distributed mappings (about 8100 fused slots), 32 times less for the register-resident thread-per-ODE mapping
 * (K+1 <= 16); a mapping that does not fit is unavailable (CKB_EUNSUPPORTED from ckb_integrate for that variant).
 */
int ckb_mech_load(const ckb_mech_desc *d, ckb_mech **out);
void ckb_mech_free(ckb_mech *m);

/*
 * ckb_mech_reserve: size the handle's work-queue order scratch for batches of up to max_batch systems (the paper's
 * "global step over all grid points"; "any scratch is sized at load time or passed by the
 * caller").  Grow-only (a smaller max_batch than what is reserved changes nothing).  Synchronises the device and
 * (re)allocates; call it between steps, never concurrently with work on the handle.  ckb_integrate refuses a batch beyond the reserved size with CKB_ECAPACITY (batches below 4096 systems need
 * no scratch).
 */
#define CKB_DEFAULT_MAX_BATCH (1 << 20)
int ckb_mech_reserve(ckb_mech *m, int64_t max_batch);

/*
 * ckb_mech_load2: ckb_mech_load for NASA fits with two temperature ranges ("thermodynamic properties are
 * typically fitted as polynomials across different temperature ranges"; reading R30, the Chemkin convention):
 *   nasa_high HOST [K][7]  a1..a7 of the high range; d->nasa is the low range
 *   T_mid     HOST [K]     species k uses nasa_high[k] where T > T_mid[k] and d->nasa[k] where T <= T_mid[k]
 * Both NULL: identical to ckb_mech_load.  The switch is taken per species and per evaluation of f(y), from the
 * temperature of the argument (a system may cross T_mid while it reacts); it is a select between two table rows, not a
 * branch.  Everything else (packing, limits, ownership, errors) as ckb_mech_load; ckb_mech_specialize generates both
 * ranges.  ckb_mech_precompile / ckb_mech_codegen / ckb_mech_pack_stats describe the one-range mechanism of `d`.
 */
int ckb_mech_load2(const ckb_mech_desc *d, const double *nasa_high, const double *T_mid, ckb_mech **out);

/*
 * ckb_mech_load3: ckb_mech_load2 (nasa_high / T_mid may both be NULL) plus pressure-dependent "fall-off" reactions
 * (P:80 refers to the Chemkin manual for the formulation; reading R31 takes that manual's form):
 *   n_falloff            number of fall-off reactions (0: identical to ckb_mech_load2)
 *   fo_reaction HOST [n] reaction index; its arr_A / arr_beta / arr_E are then the HIGH-pressure limit k_inf (A > 0)
 *   fo_low      HOST [n][3] A_0 (> 0), beta_0, E_0 (cal/mol) of the low-pressure limit k_0
 *   fo_troe     HOST [n][4] a, T***, T*, T** of Troe's broadening; a = NaN: Lindemann (F = 1); T** = +inf: the
 *                        three-parameter form (no exp(-T** / T) term); T***, T* > 0 (+inf allowed)
 *     P_r = k_0 [M] / k_inf,   k = k_inf (P_r / (1 + P_r)) F,   rate of progress = k prod C   (no further [M] factor)
 *     log10 F = log10 F_cent / (1 + ((log10 P_r + c) / (n - 0.14 (log10 P_r + c)))^2),  c = -0.4 - 0.67 log10 F_cent,
 *     n = 0.75 - 1.27 log10 F_cent,  F_cent = (1 - a) exp(-T/T***) + a exp(-T/T*) + exp(-T** / T)
 * [M] uses the reaction's third-body efficiencies if it is also listed in tb_reaction, else all alpha = 1.  On the
 * device the factor P_r/(1+P_r) F takes the place of the reaction's third-body concentration (it is a per-reaction
 * multiplier of the same kind), so the reaction loop is unchanged.  CKB_EINVAL: a reaction listed twice or out of range,
 * non-positive A_0 or A_inf, non-finite parameters.
 */
int ckb_mech_load3(const ckb_mech_desc *d, const double *nasa_high, const double *T_mid, int32_t n_falloff,
                   const int32_t *fo_reaction, const double *fo_low, const double *fo_troe, ckb_mech **out);

/* number of species / reactions / fused reaction slots / algorithmic flops per f(y) */
int ckb_mech_info(const ckb_mech *m, int32_t *n_species, int32_t *n_reactions, int32_t *n_slots,
                  double *flops_per_rhs);

/*
 * Mechanism-specialised kernels for the thread-per-ODE mapping (K+1 <= 16).  The paper generated its source-term
 * subroutines from the mechanism with a code generator and ran them one thread per system; these
 * calls are that generator: f(y) (Eq. 2-6) is written out as straight-line CUDA with every mechanism constant a
 * literal and C_k, [M], q_s in registers, compiled with the integrators by the CUDA runtime compiler (NVRTC, found
 * with dlopen; $CKB_NVRTC overrides the path) and cached on disk (<library directory>/build/jit or $CKB_JIT_CACHE).
 *
 * ckb_mech_specialize: build (or fetch from the cache) and load the specialised kernels for the current device;
 *   afterwards CKB_VARIANT_THREAD (and AUTO where it picks thread-per-ODE), ckb_rhs and the cost-proxy queue order
 *   run them instead of the table-driven kernels.  Synchronous, seconds when not cached.  Results differ from the
 *   table-driven kernels by summation order only.  CKB_EUNSUPPORTED: K+1 > 16 or NVRTC not found (the handle keeps
 *   working with the table-driven kernels); CKB_ECUDA: compilation or loading failed, text via ckb_codegen_log().
 * ckb_mech_precompile: host-only (no CUDA call): generate and compile for `arch` ("sm_100a" if NULL) into the cache.
 * ckb_mech_codegen: host-only: the generated f(y) body as text.  Copies at most cap-1 characters plus a NUL into
 *   buf (buf may be NULL when cap is 0) and stores the size needed, NUL included, in *needed.
 */
int ckb_mech_specialize(ckb_mech *m);
int ckb_mech_precompile(const ckb_mech_desc *d, const char *arch);
int ckb_mech_codegen(const ckb_mech_desc *d, char *buf, int64_t cap, int64_t *needed);
const char *ckb_codegen_log(void); /* compiler log of the calling thread's last specialize / precompile */

/*
 * Chemkin-format reader and the paper's reversible -> irreversible converter (Appendix A).
 * Host-side preprocessing, no device work.
 *   mech_text    HOST  NUL-terminated text of a mechanism file: ELEMENTS, SPECIES, [THERMO], REACTIONS blocks
 *   thermo_text  HOST  NUL-terminated text of a thermodynamic database (THERMO block), or NULL if mech_text has one
 *   fit_T3       HOST  [3] the three distinct temperatures (K) of Appendix A, or NULL for 1000, 1500, 2000 K (the paper
 *                      does not say which it used: DESIGN.md reading R33)
 * Every reversible reaction ("=" / "<=>") becomes two irreversible ones: the reverse one takes its REV parameters if
 * given, else (A_r, beta_r, E_r) from Eq. A.10-A.12 through k_r = k_f / K_c at the three temperatures, K_c in the Chemkin
 * form from the NASA fits incl. a7 (reading R32).  A reversible fall-off reaction gets a reverse fall-off reaction with
 * both limits fitted that way (P_r and F are the same for both directions).  Units are converted to mol-cm-s-K and
 * cal/mol.  Supported syntax and what is refused: see csrc/ckb_chemkin.cu.
 * ckb_chemkin_desc fills `d` and the ckb_mech_load3 arguments with pointers into the object (valid until
 * ckb_chemkin_free; the low temperature range is d->nasa, the high one *nasa_high, R30).
 * Errors: CKB_EINVAL (syntax, unknown species, unbalanced reaction, missing thermo), CKB_EUNSUPPORTED (a construct
 * outside the list above), CKB_ENOMEM; ckb_chemkin_error() returns the calling thread's last message.
 */
typedef struct ckb_chemkin ckb_chemkin;
int ckb_chemkin_parse(const char *mech_text, const char *thermo_text, const double *fit_T3, ckb_chemkin **out);
void ckb_chemkin_free(ckb_chemkin *ck);
int ckb_chemkin_desc(const ckb_chemkin *ck, ckb_mech_desc *d, const double **nasa_high, const double **T_mid,
                     int32_t *n_falloff, const int32_t **fo_reaction, const double **fo_low, const double **fo_troe);
const char *ckb_chemkin_species(const ckb_chemkin *ck, int32_t k);          /* name of species k, or NULL */
/* which reaction of the file the irreversible reaction j came from (0-based), and whether it is a generated reverse */
int ckb_chemkin_reaction_origin(const ckb_chemkin *ck, int32_t j, int32_t *input_reaction, int32_t *is_reverse);
const char *ckb_chemkin_error(void);

/*
 * ckb_integrate: advance every system i in [0, N) from t to t+dt, in place.
 *   states   DEVICE  SoA, row-major [(K+1)][ld]: row 0 = T (K), rows 1..K = mass fractions Y_k;
 *                    element (c, i) at states[c*ld + i]; ld >= N.  Caller-owned (e.g. a torch tensor).
 *   pressure DEVICE  [N] dyn/cm^2, or NULL to use p_uniform for every system (constant over the call).
 *   t, dt            f is autonomous; t only anchors the sub-step clock.  dt > 0.
 *   rtol, atol       tolerances: RKCK Eq. 16 with eps = rtol, eps*delta = atol; RKC Eq. 32.
 *   method, variant  CKB_METHOD_*, CKB_VARIANT_*.
 *   status   DEVICE  [N] int32 or NULL: CKB_ST_* per system.  A failed system holds its last accepted state.
 *   stats    DEVICE  [4][N] int32 or NULL: f(y) evaluations, accepted steps, rejected steps, largest
 *                    RKC stage count (0 for RKCK).
 *   stream           cudaStream_t as void* (NULL = legacy default stream).
 * Asynchronous on `stream`: never synchronises, allocates nothing (all scratch belongs to the handle and was sized by
 * ckb_mech_load / ckb_mech_reserve).  No state is carried from one call to the next, but calls on ONE handle
 * share that scratch (queue order; stage vectors of the thread-per-ODE variant for K+1 > 16): they must be
 * stream-ordered -- same stream, or ordered by events.  For concurrent calls on several streams load one handle per
 * stream.  N == 0 is a no-op.  Errors: CKB_EINVAL for bad arguments, CKB_ECAPACITY for N beyond the reserved batch
 * size, CKB_EUNSUPPORTED if the variant cannot hold the mechanism (the 2- / 4-lane variants need K+1 <= 16, the 8-,
 * 16- and 32-lane ones K+1 <= 14, 7 or 4 times the lanes per system, see ckb_host.h; thread-per-ODE takes any K),
 * CKB_ECUDA if the launch failed.
 */
int ckb_integrate(const ckb_mech *m, double *states, const double *pressure, double p_uniform,
                  int64_t N, int64_t ld, double t, double dt, double rtol, double atol, int32_t method,
                  int32_t variant, int32_t *status, int32_t *stats, void *stream);

/*
 * ckb_integrate_static: ckb_integrate for callers that must never allocate device memory on the call path (code under
 * CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc): the work-queue order scratch does not
 * come from the handle but from ONE file-scope device array inside the library (csrc/ckb_order.cu), 12 bytes per system
 * + 8 KB = 6.0 MiB for CKB_STATIC_MAX_BATCH systems, which every GPU that loads the library holds until the process
 * exits.  Arguments, layouts, results and status codes exactly as ckb_integrate (constant-pressure closure); the call
 * and everything behind it use no cudaMalloc, cudaFree or allocating library routine.
 * N > CKB_STATIC_MAX_BATCH is refused with CKB_ECAPACITY (nothing is launched).
 * The array is shared by EVERY call in the process (all handles, all streams) and keeps the last call's contents (the
 * part that must start at zero is cleared on `stream` by each call): two calls that overlap on the GPU race on it and
 * may skip systems or advance them twice -- order them (same stream, or events).  ckb_integrate itself does not use it.
 */
#define CKB_STATIC_MAX_BATCH 524288
int ckb_integrate_static(const ckb_mech *m, double *states, const double *pressure, double p_uniform, int64_t N,
                         int64_t ld, double t, double dt, double rtol, double atol, int32_t method, int32_t variant,
                         int32_t *status, int32_t *stats, void *stream);

/*
 * ckb_integrate_host: the same call with HOST buffers (states, pressure, status, stats as above but in
 * host memory, pinned or pageable).  Copies host->device, integrates, copies device->host on `stream`
 * and synchronises it before returning -- the per-global-step protocol the paper timed.  Uses
 * a grow-only device workspace owned by the handle (not thread-safe per handle).
 */
int ckb_integrate_host(ckb_mech *m, double *states, const double *pressure, double p_uniform, int64_t N,
                       int64_t ld, double t, double dt, double rtol, double atol, int32_t method,
                       int32_t variant, int32_t *status, int32_t *stats, void *stream);

/*
 * Constant-volume closure (the other operator-split chemistry mode; P:243 names it without equations, DESIGN.md
 * reading R29 takes the textbook form): the density rho of each system is given and constant over the call,
 *     C_k = rho Y_k / W_k,    dY_k/dt = W_k omega_k / rho                       (Eq. 2-5 unchanged)
 *     rho c_v dT/dt = - sum_k u_k omega_k W_k,   u_k = h_k - Ru T / W_k,   c_v = c_p - Ru sum_k Y_k / W_k
 * and the pressure follows from the ideal-gas law.  ckb_integrate_cv / ckb_integrate_host_cv / ckb_rhs_cv are
 * ckb_integrate / ckb_integrate_host / ckb_rhs with `density` (DEVICE resp. HOST [N], g/cm^3, or NULL to use
 * rho_uniform > 0) in place of the pressure; every other argument, the layouts, the mapping variants, the
 * asynchrony and the error behaviour are the same.  The same kernel templates run (the closure is a compile-time parameter).
 */
int ckb_integrate_cv(const ckb_mech *m, double *states, const double *density, double rho_uniform, int64_t N,
                     int64_t ld, double t, double dt, double rtol, double atol, int32_t method, int32_t variant,
                     int32_t *status, int32_t *stats, void *stream);
int ckb_integrate_host_cv(ckb_mech *m, double *states, const double *density, double rho_uniform, int64_t N,
                          int64_t ld, double t, double dt, double rtol, double atol, int32_t method,
                          int32_t variant, int32_t *status, int32_t *stats, void *stream);

/*
 * ckb_rhs: evaluate the source term f(y) (Eq. 2-6) once for each of N systems, without integrating;
 * dydt DEVICE [(K+1)][ld] receives (dT/dt, dY_k/dt).  Same layout and mapping variants as
 * ckb_integrate.  Used by the parity tests of the source term and by the roofline measurement.
 * `repeat` >= 1 evaluates f that many times per system inside the kernel (timing aid; result unchanged).
 */
int ckb_rhs(const ckb_mech *m, const double *states, const double *pressure, double p_uniform, int64_t N,
            int64_t ld, double *dydt, int32_t variant, int32_t repeat, void *stream);
int ckb_rhs_cv(const ckb_mech *m, const double *states, const double *density, double rho_uniform, int64_t N,
               int64_t ld, double *dydt, int32_t variant, int32_t repeat, void *stream);

/*
 * ckb_fp64_probe: roofline denominator.  Runs a register-resident kernel of independent DFMA chains on
 * every SM (iters FMAs per chain) on `stream`, times it with CUDA events and returns the achieved
 * FP64 rate in FLOP/s (2 per FMA) in *flops_per_s.  kind 0 = DFMA chains; kind 1 = exp(double) calls
 * (returns exp evaluations per second).  Synchronises `stream`.
 */
int ckb_fp64_probe(int32_t kind, int64_t iters, double *per_second, void *stream);

/*
 * ckb_mech_pack_stats: host-only (no CUDA call).  Validates `d`, packs it for `lanes` lanes per system
 * (1, 2, 4, 8, 16 or 32) and reports the packing: stats[0] fused reaction slots, [1] slot rounds per f(y),
 * [2] gather steps per f(y), [3] shared-memory bank-conflict replays left in the gather per f(y) after
 * scheduling (lanes = 32 only, else 0), [4] the same for the concentration reads, [5] table size in
 * 8-byte words, [6] shared-memory doubles per system, [7] register slots per lane (NV).
 */
int ckb_mech_pack_stats(const ckb_mech_desc *d, int32_t lanes, int32_t *stats8);

const char *ckb_strerror(int code);
const char *ckb_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* CKB_H_ */
