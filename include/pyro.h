/* pyro.h -- C ABI of libpyro: per-point combustion thermochemistry on one NVIDIA B200 (sm_100a).
 *
 * The data-parallel hot path of Pyrometheus (arXiv 2503.24286, Appendix A; citations are
 * PAPER.md:LINE of the extracted paper text):
 *   - NASA-7 species thermodynamics                          (A.11)-(A.13), (A.31)
 *   - Newton inversion of temperature from internal energy   (A.25)-(A.30)
 *   - net production rates  omega_i = sum_j nu_ij R_j        (A.5)-(A.10)
 *     with Arrhenius, third-body, Lindemann/Troe falloff rate coefficients
 *     and reverse rates from equilibrium constants           (A.10)
 *
 * Conventions
 *   Units: SI with kmol. W kg/kmol, C kmol/m^3, omega kmol/(m^3 s), e J/kg, T K, rho kg/m^3,
 *          R = 8314.46261815324 J/(kmol K), p0 = 101325 Pa.
 *   Fields: FP64, structure of arrays [species][points]: species k of point p is X[k*ld + p],
 *          ld >= n in doubles.  "device" pointers are CUDA device memory on the mechanism's
 *          device; "host" pointers are ordinary (preferably pinned) host memory.
 *   Every function returns a pyro_status (0 = PYRO_OK); nothing throws or aborts across the ABI.
 *   Device calls enqueue on `cuda_stream` (a cudaStream_t passed as void*, NULL = default
 *   stream) and return without synchronising; they allocate nothing and copy nothing.
 *   Concurrent calls on one handle from several host threads are allowed.
 *   There is no CPU fallback: without a CUDA device pyro_mech_create fails with PYRO_ERR_CUDA.
 *   Environment variables read by pyro_mech_create are TEST HOOKS that force a launch shape the library would
 *   not choose by itself (they exist so that the parity tests reach every kernel variant); they are not part of
 *   the interface and change no result: PYRO_TABLES=shared|global, PYRO_RATES_BLOCK=<threads>,
 *   PYRO_B_PLANE=shared, PYRO_CARVEOUT=<percent>, PYRO_RATES_POINTS=1|2 (grid points per thread of the rates kernel), PYRO_RATES_TWO_BLOCKS=0|1, PYRO_PACK_SINGLES=0|1,
 *   PYRO_HOST_SLAB=<points> (pyro_source_terms_host), PYRO_JAC_KERNEL=point|block (the one-thread-per-point / the block-cooperative Jacobian kernel), PYRO_JAC_V_PLANE=shared, PYRO_JAC_BLOCK=<threads>, PYRO_JAC_EXT=global
 *   (pyro_get_jacobian), PYRO_CN_BLOCK=32|64 (points per block of the Crank-Nicolson LU kernel; read once per process at the first Crank-Nicolson call; 64 only up to 97 species), PYRO_DEBUG=1 (prints the launch shape to stderr).
 */
#ifndef PYRO_H
#define PYRO_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    PYRO_OK = 0,
    PYRO_ERR_NULL = 1,        /* a required pointer is NULL                                         */
    PYRO_ERR_BAD_SIZE = 2,    /* n < 0, ld < n, n_species < 1, n_reactions < 0, max_iter < 1 ...     */
    PYRO_ERR_BAD_MECH = 3,    /* index out of range, A <= 0, W <= 0, bad Troe temperature,
                                 coefficient <= 0, more than 3 molecules on a side, CSR not monotone,
                                 unknown reaction type                                              */
    PYRO_ERR_TOO_LARGE = 4,   /* species / reactions beyond what the on-chip staging can hold (255 species) */
    PYRO_ERR_ALIGN = 5,       /* a field pointer is not 8-byte aligned                               */
    PYRO_ERR_CUDA = 6,        /* CUDA runtime error (text via pyro_last_error_string)                */
    PYRO_ERR_UNSUPPORTED = 7  /* valid input that this build cannot evaluate (see PYRO_T_MIN / PYRO_T_MAX)  */
} pyro_status;

/* Supported temperature range of the rates (K).  pyro_mech_create examines the mechanism over this range
 * and refuses (PYRO_ERR_UNSUPPORTED) one whose rates it could not evaluate in FP64 there -- see
 * pyro_get_net_production_rates.  Outside the range nothing is checked. */
#define PYRO_T_MIN 250.0
#define PYRO_T_MAX 6000.0

/* reaction types */
enum { PYRO_ELEMENTARY = 0, PYRO_THREE_BODY = 1, PYRO_FALLOFF_LINDEMANN = 2, PYRO_FALLOFF_TROE = 3 };

typedef struct pyro_mech pyro_mech; /* opaque; owns the device tables of one mechanism on one device */

/* Host description of a mechanism.  All pointers are HOST memory, borrowed only for the
 * duration of pyro_mech_create (the caller may free everything afterwards).
 * Reaction j reads  sum_i nu'_ij S_i <=> sum_i nu''_ij S_i  (A.4) PAPER.md:903. */
typedef struct {
    int32_t n_species, n_reactions, n_elements; /* n_elements may be 0                             */
    const double *mol_weight;                   /* [n_species] kg/kmol, > 0                        */
    const double *nasa_lo, *nasa_hi;            /* [n_species][7] a1..a7 for T < T_mid / T >= T_mid */
    const double *t_mid;                        /* [n_species] K                                   */
    const int32_t *elem_comp;                   /* [n_species][n_elements] or NULL; if given, every
                                                   reaction must be element balanced              */
    const int32_t *reac_ptr, *reac_species, *reac_coeff; /* CSR of nu' : ptr[n_reactions+1]       */
    const int32_t *prod_ptr, *prod_species, *prod_coeff; /* CSR of nu''                           */
    const double *A, *b, *theta; /* [n_reactions] k = A T^b exp(-theta/T) (A.9): A > 0 in
                                    (m^3/kmol)^(order-1)/s, theta = Ea/R in K (any sign);
                                    for falloff reactions this is the high-pressure limit          */
    const uint8_t *type;         /* [n_reactions] PYRO_ELEMENTARY ... PYRO_FALLOFF_TROE            */
    const uint8_t *reversible;   /* [n_reactions] 1: reverse rate from K_c (A.10); 0: r_r = 0      */
    const double *eff_default;   /* [n_reactions] default third-body efficiency (usually 1)        */
    const int32_t *eff_ptr, *eff_species; /* CSR of non-default efficiencies: ptr[n_reactions+1];
                                             within a reaction in any order, each species at most once */
    const double *eff_value;
    const double *A0, *b0, *theta0; /* [n_reactions] low-pressure limit, read when type >= 2       */
    const double *troe; /* [n_reactions][4] alpha, T***, T*, T** read when type == 3;
                           T* or T** = +inf drops that term (3-parameter form when T** = +inf)     */
} pyro_mech_desc;

/* Validate `desc`, flatten it into device tables (per-species Gibbs rows, packed Arrhenius
 * coefficients, fixed-width species slots, efficiency lists, falloff parameters, NASA energy tables) and
 * upload them to CUDA device `device`.  *out receives the handle.  On error *out = NULL. */
int pyro_mech_create(const pyro_mech_desc *desc, int device, pyro_mech **out);

/* Free the device tables.  pyro_mech_destroy(NULL) is a no-op returning PYRO_OK.  The caller
 * must make sure no launch that uses the handle is still running. */
int pyro_mech_destroy(pyro_mech *mech);

/* Newton controls of pyro_get_temperature: stop when |dT| < abs_tol_K after the update,
 * at most max_iter iterations.  Defaults 1e-6 K and 10 (BASELINE.json configs[4]).  May be called while other
 * threads enqueue on the handle: a call enqueued concurrently uses either the old or the new pair member-wise. */
int pyro_mech_set_newton(pyro_mech *mech, double abs_tol_K, int max_iter);

/* Temperature from internal energy: solves  sum_k Y_k e_k(T) = e  per point by Newton's
 * method, T <- T - (Y.e(T) - e)/c_v(T,Y)   (A.25)-(A.30) PAPER.md:1008-1029, listing 22 :672.
 *   rho      [n]            device, may be NULL (the ideal-gas caloric EOS does not use it)
 *   e        [n]            device, J/kg
 *   Y        [n_species][ld] device, mass fractions (not clipped, not renormalised)
 *   T_guess  [n]            device, K, > 0
 *   T        [n]            device, out; may alias T_guess
 *   n_not_converged         device int32 (4-byte aligned) or NULL: incremented once per point that hit max_iter
 *                           (the last iterate is still written; this is not an error)
 * n == 0 returns PYRO_OK and launches nothing. */
int pyro_get_temperature(const pyro_mech *mech, int64_t n, int64_t ld, const double *rho, const double *e,
                         const double *Y, const double *T_guess, double *T, int32_t *n_not_converged,
                         void *cuda_stream);

/* Enthalpy form of the inversion ("minor modifications"; `do_energy=False` of listing
 * 22): solves  sum_k Y_k h_k(T) = h  per point, T <- T - (Y.h(T) - h)/c_p(T,Y).
 * Arguments, stop rule and non-convergence report as pyro_get_temperature, with h [n] in J/kg. */
int pyro_get_temperature_from_enthalpy(const pyro_mech *mech, int64_t n, int64_t ld, const double *h,
                                       const double *Y, const double *T_guess, double *T,
                                       int32_t *n_not_converged, void *cuda_stream);

/* Ideal-gas equation of state (A.2)-(A.3) PAPER.md:892-899:  p = rho R T / W,  W = (sum_k Y_k/W_k)^-1.
 *   pyro_get_density :  rho[p] = p[p] W / (R T[p])      pyro_get_pressure :  p[p] = rho[p] R T[p] / W
 * All pointers device; p / rho / T [n], Y [n_species][ld]; the output may alias its scalar input. */
int pyro_get_density(const pyro_mech *mech, int64_t n, int64_t ld, const double *p, const double *T,
                     const double *Y, double *rho, void *cuda_stream);
int pyro_get_pressure(const pyro_mech *mech, int64_t n, int64_t ld, const double *rho, const double *T,
                      const double *Y, double *p, void *cuda_stream);

/* Net molar production rates omega[k*ld+p] = sum_j nu_kj R_j  (A.5)-(A.10) PAPER.md:908-934 from
 *   rho [n], T [n], Y [n_species][ld]   (device; T > 0, rho > 0, Y >= 0 are preconditions)
 *   omega [n_species][ld]               (device, out; must not overlap Y)
 * Range.  The kernel evaluates (A.7), (A.10) from one factor E_k = exp(g_k/RT - lambda_k(T)) RT/p0 per species
 * and point, 1/K_c,j = prod_prod E_k / prod_reac E_k, where lambda_k(T) is the part of g_k/RT that every
 * reversible reaction conserves (it cancels exactly in K_c; chosen at create time so that the E_k stay
 * near 1).  Products of these factors must stay inside FP64 (2^+-1022) although K_c itself only holds their
 * ratio.  pyro_mech_create therefore evaluates log2 E_k at 64 temperatures over [PYRO_T_MIN, PYRO_T_MAX]:
 * a reaction whose per-side sums stay below 700 is evaluated side by side (fast path); any other reaction is
 * evaluated in reactant/product pairs, whose partial products end at 1/K_c; and the call returns
 * PYRO_ERR_UNSUPPORTED if even those partial sums exceed 900 (K_c within a factor 2^120 of the FP64 limits), or if
 * log2 of a rate coefficient exceeds 2^30 in magnitude.  Inside the supported range the rates are thus finite
 * wherever the definition's own K_c and rate coefficients are -- never a silent NaN. */
int pyro_get_net_production_rates(const pyro_mech *mech, int64_t n, int64_t ld, const double *rho,
                                  const double *T, const double *Y, double *omega, void *cuda_stream);

/* The whole source-term step in ONE launch (the source terms "for a given
 * density, mass fractions, and internal energy"): per point the Newton solve of pyro_get_temperature from
 * (e, Y, T_guess), then the production rates at that temperature.  All pointers device:
 *   rho, e, T_guess [n], Y [n_species][ld]  in;   T [n] (may alias T_guess), omega [n_species][ld] (must not overlap Y)  out;
 *   n_not_converged as in pyro_get_temperature.
 * Results are those of pyro_get_temperature followed by pyro_get_net_production_rates (same iterates, same rates). */
int pyro_source_terms(const pyro_mech *mech, int64_t n, int64_t ld, const double *rho, const double *e,
                      const double *Y, const double *T_guess, double *T, double *omega, int32_t *n_not_converged,
                      void *cuda_stream);

/* Batched reactor march: one adiabatic isochoric reactor (A.1) PAPER.md:886-888 per point,
 *     rho dY_k/dt = W_k omega_k(rho, T, Y),   rho and e constant,   T from (e, Y) by the Newton solve of pyro_get_temperature,
 * advanced by n_steps classical fourth-order Runge-Kutta steps of size dt (s) in ONE launch, the state
 * staying on chip across the stages.  All pointers device:
 *   rho, e [n]            in
 *   Y [n_species][ld]     in: initial mass fractions; out: mass fractions after n_steps steps (not clipped, not renormalised)
 *   T [n]                 in: Newton starting guess; out: temperature of the final state
 *   work [n_species][ld]  scratch (contents undefined afterwards); must not overlap Y
 *   n_not_converged       as in pyro_get_temperature: incremented once per Newton solve (4 per step + 1) that hit the cap
 * Every stage starts its Newton iteration from the temperature of the stage before.  The step is the caller's: the
 * scheme is explicit and unstable beyond the chemical time scale (the paper's H2 case needs 10 ns). n_steps = 0 only
 * inverts the temperature. */
int pyro_reactor_rk4(const pyro_mech *mech, int64_t n, int64_t ld, const double *rho, const double *e, double *Y,
                     double *T, double dt, int32_t n_steps, double *work, int32_t *n_not_converged, void *cuda_stream);

/* pyro_reactor_rk4 for callers that cannot allocate device memory -- and so have no `work` field to pass.  That is the
 * situation of code running inside somebody else's memory budget: a solver plug-in whose host application owns every
 * byte of the GPU and hands out only the state arrays, a call made while the application's memory pool is frozen
 * (between its set-up phase and its tear-down), a real-time or in-situ loop in which cudaMalloc's implicit device
 * synchronisation is not acceptable.  Same march, same results as pyro_reactor_rk4; the scratch it needs (the running
 * sum of the stage slopes, one double per species and reactor, and the launch's work counter) is a fixed array built
 * into the library image instead.  The call itself performs no cudaMalloc / cudaFree and calls nothing that does.
 *   Limit.   n_species * (n rounded up to a multiple of 32) <= PYRO_RK4_STATIC_MAX_DOUBLES (4 Mi doubles = 32 MiB:
 *            79 136 reactors of a 53-species mechanism, 466 016 of a 9-species one); beyond it the call returns
 *            PYRO_ERR_TOO_LARGE and launches nothing -- march the batch in slabs.  `ld` does not enter the limit.
 *   Cost.    every GPU on which the process uses libpyro holds those 32 MiB (+ 256 bytes) from the moment the
 *            library is loaded there until the process exits, whether or not this function is ever called.
 *   First call on a device.  Looks up the array's address on that device and raises the kernel's shared-memory
 *            limit (two cheap, non-allocating runtime queries; later calls skip them).  Make that first call
 *            outside any stream capture; n_steps = 0 on one reactor is enough.
 *   Sharing. There is ONE array per device, used by every call on every handle and stream.  Two calls whose kernels
 *            may run at the same time on one device (different streams without an event between them, or two host
 *            threads) race on it and both results are garbage: keep the calls of a device on one stream or order them
 *            yourself.  Nothing in the array has to survive between calls and nothing in it is read before this call
 *            has written it (the work counter is reset on `cuda_stream` first), so stale contents are harmless.
 * Arguments, preconditions and n_not_converged exactly as pyro_reactor_rk4, minus `work`. */
#define PYRO_RK4_STATIC_MAX_DOUBLES 4194304
int pyro_reactor_rk4_static(const pyro_mech *mech, int64_t n, int64_t ld, const double *rho, const double *e, double *Y,
                            double *T, double dt, int32_t n_steps, int32_t *n_not_converged, void *cuda_stream);

/* Implicit march of the same reactors (second half): Crank-Nicolson (A.32) PAPER.md:1043-1062,
 *     Y^{m+1} - Y^m - dt/2 (s^{m+1} + s^m) = 0,   s_k = W_k omega_k / rho,
 * each step solved by `newton_iters` Newton iterations (A.33)-(A.35) started from Y^m, with the analytic Jacobian
 * (A.36) at fixed (rho, e) (pyro_get_jacobian, PYRO_JAC_FIXED_E) and a dense LU per point without pivoting (the matrix
 * is I - dt/(2 rho) J).  The iteration count is fixed (data-independent control flow, no host synchronisation): a launch
 * sequence of the library's own temperature, rates and Jacobian kernels plus the per-point linear algebra, all on
 * `cuda_stream`.  Arguments as pyro_reactor_rk4, and
 *   update_tol       a point whose last Newton update max_k |dY_k| of a step is not below it (or not finite) is counted
 *   work             device scratch of *doubles doubles as pyro_reactor_cn_work_doubles(mech, ld, &doubles) reports; must not overlap Y
 *   n_not_converged  += temperature solves that hit their cap + (point, step) pairs counted by update_tol
 * Mechanisms of more than 127 species: PYRO_ERR_UNSUPPORTED.
 * Step-size regime of the LU.  The elimination takes the pivots in the given order and inverts them without a magnitude
 * check.  That is safe while I - dt/(2 rho) J is diagonally dominated and has been verified beyond it, against an
 * elimination with partial pivoting, up to |dt/(2 rho) J|_inf = 10 (100 times the explicit stability step; no reactor
 * of the test batches lost a digit there).  Above that regime element growth is neither bounded nor detected as such: the
 * only report is n_not_converged (a non-finite or too large last update), so march stiffer steps with a tolerance that
 * means something, or in several smaller steps. */
int pyro_reactor_cn_work_doubles(const pyro_mech *mech, int64_t ld, int64_t *doubles);
int pyro_reactor_cn(const pyro_mech *mech, int64_t n, int64_t ld, const double *rho, const double *e, double *Y,
                    double *T, double dt, int32_t n_steps, int32_t newton_iters, double update_tol, double *work,
                    int32_t *n_not_converged, void *cuda_stream);

/* Chemical Jacobian (eq. (6); (A.36) PAPER.md:1057) of the source terms S_i = W_i omega_i
 * ((A.1) PAPER.md:888), analytic:
 *   J[(i*n_species + k)*ld + p] = dS_i/dY_k     [n_species*n_species][ld], device, out; must not overlap Y
 *   dSdT[i*ld + p]              = dS_i/dT at fixed (rho, Y)   [n_species][ld], device, out, or NULL
 * from rho [n], T [n], Y [n_species][ld] as in pyro_get_net_production_rates.  The mass fractions are independent
 * variables (no sum-to-one constraint is applied), C_k = rho Y_k / W_k (A.8).  `mode` says what is held fixed
 * while Y_k varies:
 *   PYRO_JAC_FIXED_T   rho and T:  J_ik = W_i (rho/W_k) sum_j nu_ij dR_j/dC_k
 *   PYRO_JAC_FIXED_E   rho and the internal energy e (an adiabatic isochoric reactor (A.1); what the paper's listing 23
 *                      differentiates, through the temperature inversion):  J_ik - dS_i/dT e_k(T)/c_v(T,Y)
 * The derivatives of the third-body and Lindemann / Troe forms are included (through [M] and through T).
 * Mechanisms of more than 127 species: PYRO_ERR_UNSUPPORTED.  The limit is the tensor memory of an SM: per species row the
 * kernel keeps two FP64 accumulators for each of a warp's points (the column dS_i/dY_k being built and dS_i/dT), four of the
 * 512 columns a block can hold, so 127 species + the [M] row fill it; the rates path needs half of that and goes to 255.
 * (The dense output is 8 n_species^2 bytes per point -- 131 KB at 128 species -- so larger mechanisms want a sparse
 * output format before they want a larger kernel.)  Launches on one handle share a scratch buffer and are ordered after
 * one another (also across streams). */
enum { PYRO_JAC_FIXED_T = 0, PYRO_JAC_FIXED_E = 1 };
int pyro_get_jacobian(const pyro_mech *mech, int64_t n, int64_t ld, const double *rho, const double *T,
                      const double *Y, int mode, double *J, double *dSdT, void *cuda_stream);

/* Mixture-averaged transport properties, Appendix A.2 as printed, from
 * polynomial fits in ln T that the caller supplies (the paper takes them from Cantera):
 *   mu_k = sqrt(T) (sum_m visc[k][m] (ln T)^m)^2 (A.22)      kappa_k = sqrt(T) sum_m cond[k][m] (ln T)^m (A.24)
 *   D_kj = sqrt(T) sum_m diff[k][j][m] (ln T)^m (A.19), m = 0..4; no pressure factor is applied (the fits are at the
 *   caller's pressure); the diagonal diff[k][k] is never read.
 * pyro_get_transport evaluates, per point, the Wilke mixture viscosity (A.20)-(A.21), the mixture conductivity
 * (A.23) and the mixture-averaged diffusivities (A.18) with mole fractions X_k = W Y_k/W_k (A.3):
 *   T [n], Y [n_species][ld]                         device, in
 *   mu [n] (Pa s), kappa [n] (W/(m K)), D [n_species][ld] (m^2/s)    device, out; D must not overlap Y
 * (A.18) is singular for a pure species (0/0): at least two species present is a precondition; T > 0.
 * The description is HOST memory, borrowed during pyro_transport_create only.  Same status codes and error text
 * (pyro_last_error_string) as the rest of the library; no CPU fallback. */
typedef struct pyro_transport pyro_transport;
typedef struct {
    int32_t n_species;
    const double *mol_weight; /* [n_species] kg/kmol                     */
    const double *visc;       /* [n_species][5]                          */
    const double *cond;       /* [n_species][5]                          */
    const double *diff;       /* [n_species][n_species][5]               */
} pyro_transport_desc;
int pyro_transport_create(const pyro_transport_desc *desc, int device, pyro_transport **out);
int pyro_transport_destroy(pyro_transport *tr);
int pyro_get_transport(const pyro_transport *tr, int64_t n, int64_t ld, const double *T, const double *Y, double *mu,
                       double *kappa, double *D, void *cuda_stream);

/* The whole source-term step from HOST buffers: (rho, e, Y, T_guess) -> (T, omega).  Copies the
 * inputs to the device in slabs of points, runs the temperature solve and the rates kernel on
 * each slab and copies T and omega back, the three stages overlapped on separate streams.
 * All pointers are host memory (pinned memory gives asynchronous copies); layouts as above
 * with leading dimension `ld`.  Blocks until the results are in T and omega.
 * *n_not_converged (host, may be NULL) receives the Newton non-convergence count. */
int pyro_source_terms_host(pyro_mech *mech, int64_t n, int64_t ld, const double *rho, const double *e,
                           const double *Y, const double *T_guess, double *T, double *omega,
                           int64_t *n_not_converged);

/* Facts about a packed mechanism, for reports: fills up to `cap` int64 values
 *   [0] n_species  [1] n_reactions  [2] reactions in the plain class  [3] in the extended class
 *   [4] table bytes  [5] 1 if the rates kernel stages the tables in shared memory, 0 if it reads
 *   them from global memory  [6] threads per block of the rates kernel (points per block: [6] x [12])
 *   [7] dynamic shared memory per block (bytes)  [8] resident (persistent) blocks per SM
 *   [9] registers per thread of the rates kernel  [10] local (spill) bytes per thread
 *   [11] SM count of the device  [12] grid points per thread of the rates kernel
 *   (1; 2 for small mechanisms: the two-points-per-thread kernel)
 *   [13] tensor-memory columns a block allocates  [14] 1 if B_k = 1/E_k is kept in tensor memory
 *   beside omega_k (else in a second shared-memory plane)
 * returns the number of values written (negative pyro_status on error). */
int pyro_mech_info(const pyro_mech *mech, int64_t *out, int cap);

/* Measures the FP64 FMA peak of `device`: independent DFMA chains on every SM for about
 * `millis` ms; *tflops = 2 * FMAs / time.  Used as the roofline denominator cross-check. */
int pyro_probe_fp64_peak(int device, double millis, double *tflops);

/* Probes behind two design decisions (`python bench.py --probes` prints them):
 * pyro_probe_dmma_peak: sustained rate of the FP64 tensor-core instruction mma.sync.m8n8k4.f64 (8 independent
 *   accumulators per warp, every SM) for about `millis` ms; *tflops = 2 flops per multiply-add.
 * pyro_probe_indexed_rmw: one block of `warps_per_sm` warps (1..8) per SM; every thread performs, per iteration, sixteen
 *   independent read-modify-writes of a double at pseudo-random warp-uniform slots out of 64, in shared memory
 *   (mode 0), in tensor memory with tcgen05.ld / wait / add / tcgen05.st / wait (mode 1), or only the tensor-memory
 *   loads (mode 2); *cycles_per_iteration = SM clock cycles per iteration of block 0. */
int pyro_probe_dmma_peak(int device, double millis, double *tflops);
int pyro_probe_indexed_rmw(int device, int warps_per_sm, int mode, double *cycles_per_iteration);

const char *pyro_status_string(int status); /* static text for a pyro_status                       */
const char *pyro_last_error_string(void);   /* detail of the last error on this thread (may be "") */

#ifdef __cplusplus
}
#endif
#endif /* PYRO_H */
