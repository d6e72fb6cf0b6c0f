/* ck.h -- C ABI of the B200-native batched reactor integration library (libck.so).
 *
 * The operations are those of arXiv 1608.05794 (Stone, Alferman, Niemeyer); citations are
 * PAPER.md:<line> of the reference text plus the equation / algorithm they fall in.
 *
 * Problem statement: n independent constant-pressure homogeneous reactors,
 * state y = [T, Y_1..Y_K] (N = K+1 components), each advanced over one operator-split CFD step dt.
 *
 * CONVENTIONS
 *   units     cgs-mol-K; activation energies in cal/mol; pressure in dyn/cm^2 (1 atm = 1.01325e6).
 *   layout    batches are component-major FP64: y[c*ld + r], c = 0 is T, c = 1..K is Y_k, r < n <= ld.
 *   pointers  every `y`, `p`, `dydt`, `J`, `n_accept`, `n_reject`, `status`, `h_last`, `ws` argument of the
 *             non-_host entry points is a DEVICE pointer owned by the caller (e.g. a torch tensor);
 *             `ck_mech_desc`, `ck_opts`, `ck_report` are HOST structs.  The *_host entry points take HOST
 *             pointers for the batch arrays and do the transfers themselves.
 *   stream    work is enqueued on the caller's stream (a cudaStream_t passed as void*; NULL = default
 *             stream).  ck_rhs / ck_jac return without synchronising.  ck_integrate_* synchronise the
 *             stream before returning when a non-NULL ck_report is passed (the counters are read back).
 *   errors    every call returns int32: CK_OK or a CK_E* code; ck_last_error() gives a thread-local
 *             message.  No exceptions, no exit().  There is NO CPU fallback: without a CUDA device the
 *             compute entry points return CK_ECUDA.
 *   ownership the library owns only the ck_mech handle (device copies of the packed mechanism).
 */
#ifndef CK_H_
#define CK_H_
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { CK_OK = 0, CK_EINVAL = 1, CK_ECUDA = 2, CK_EWORKSPACE = 3, CK_EUNSUPPORTED = 4 };
enum { CK_OP_ROS = 0, CK_OP_RKF45 = 1, CK_OP_JAC = 2 };                 /* ck_workspace_bytes `op` */
enum { CK_PLAIN = 0, CK_THREE_BODY = 1, CK_LINDEMANN = 2, CK_TROE = 3 }; /* ck_mech_desc.type */
enum { CK_JAC_ANALYTIC = 0, CK_JAC_FD = 1 };
enum { CK_CONST_PRESSURE = 0, CK_CONST_VOLUME = 1 };                    /* ck_mech_set_reactor `kind` */
/* per-reactor status written by ck_integrate_* */
enum { CK_ST_OK = 0, CK_ST_MAX_STEPS = 1, CK_ST_H_UNDERFLOW = 2, CK_ST_NONFINITE = 3, CK_ST_ZERO_PIVOT = 4 };

typedef struct ck_mech ck_mech; /* opaque */

/* Kinetic model (the paper's "binary database" of create_rate_subs, replaced by this
 * plain description).  All pointers are HOST pointers, copied at load.  Species k has NASA-7
 * coefficients a1..a7 for T <= t_mid[k] (nasa_lo) and T > t_mid[k] (nasa_hi) (Eq. 19).
 * Reaction i: sum nu'_ki X_k <=> sum nu''_ki X_k with integer coefficients in CSR form; forward rate
 * A T^beta exp(-Ea/(R T)) (Eq. 15); reverse rate from the equilibrium constant
 * (Eq. 16-18) when reversible[i] != 0, else 0.  type[i] selects the factor c_i of
 * Eq. 14: 1, [M]_i, or the Lindemann / Troe falloff form with low-pressure limit
 * (A0, beta0, Ea0) and Troe parameters (a, T***, T*, T**; T** < 0 means the term is absent).
 * Third-body efficiencies default to 1; non-unit ones are listed in CSR form (eff_*). */
typedef struct {
  int32_t struct_size; /* = sizeof(ck_mech_desc) */
  int32_t n_species, n_reactions, n_elements;
  const double* mol_wt;     /* [K] g/mol */
  const int32_t* elem_comp; /* [K*E] or NULL (only used to validate reaction balance) */
  const double *nasa_lo, *nasa_hi, *t_mid; /* [K*7], [K*7], [K] */
  const int32_t *reac_ptr, *reac_spec, *reac_nu; /* CSR nu'  : ptr[R+1], spec[], nu[] */
  const int32_t *prod_ptr, *prod_spec, *prod_nu; /* CSR nu'' */
  const double *A, *beta, *Ea;                   /* [R] */
  const uint8_t *reversible, *type;              /* [R] */
  const double *A0, *beta0, *Ea0;                /* [R] (read for falloff rows only) */
  const double* troe;                            /* [R*4] (read for Troe rows only) */
  const int32_t *eff_ptr, *eff_spec;             /* CSR non-unit efficiencies: ptr[R+1], spec[] */
  const double* eff_val;
} ck_mech_desc;

/* Solver options (Algorithm 1; the paper leaves the controller unspecified, see
 * DESIGN.md reading G8).  h0 = 0 requests the EstimateH0 rule; max_steps <= 0 means 100000. */
typedef struct {
  int32_t struct_size; /* = sizeof(ck_opts) */
  int32_t jac_mode;    /* CK_JAC_ANALYTIC | CK_JAC_FD (ROS4 only; FD: PAPER.md:281) */
  double rtol, atol;
  double h0;
  int32_t max_steps;
  int32_t flags;       /* bit 0: disable the divergence-control layer (static reactor -> lane / CTA mapping, the paper's
                          layout; for comparison).  RKF45, bit 1: lane refill only, no cooperative finisher; bits 4 / 5
                          (measurement of the finishers): every reactor counts as a straggler after the classification
                          pass / the stragglers run on the narrow finisher instead of the wide one.
                          ROS4, bit 2: force the fused CTA-per-reactor kernel, bit 3: force the batched rounds
                          (default: rounds for n >= 16384 reactors of a model with 33 <= N <= 128, analytic Jacobian),
                          bit 6 (measurement): the rounds evaluate a fresh Jacobian for EVERY attempt; by default they keep
                          f(y_n) and J(y_n) across a rejected attempt (y_n has not moved: same values, fewer evaluations,
                          so jac_evals <= attempts and rhs_evals = 2 attempts + jac_evals + 2 n). */
} ck_opts;

/* Batch totals and divergence statistics, filled on the HOST after the call (may be NULL).
 * simt_efficiency: RKF45 -- active lane-slots / issued lane-slots of the step-attempt loop (device counters).
 * ROS4, batched rounds -- slots holding an active reactor / lanes launched, summed over the kernels of all rounds
 * (counted per launch from the device-side active count).  ROS4, fused kernel -- the ANALYTIC lane utilisation of its
 * cooperative loops, (R / ceil_G(R) + N / ceil_G(N)) / 2 for CTAs of G lanes (not a counter; the measured warp
 * execution efficiency is in profiles/).  waste_p32 = Eq. 20 at width P = 32 for the static reactor->lane
 * mapping, computed from the per-reactor attempt counts (what the paper's layout would have wasted). */
typedef struct {
  int64_t attempts, accepted, rejected, rhs_evals, jac_evals, lu_factor;
  double simt_efficiency, waste_p32;
  int32_t rounds; /* re-batching rounds: attempt rounds of the batched ROS4 (+1 for its tail), 1 or 2 kernels otherwise */
  int32_t n_failed;
} ck_report;

const char* ck_last_error(void);
int32_t ck_version(void);

/* Validate and pack the mechanism (SoA, reactions grouped by type, reverse-rate polynomial folded per
 * temperature interval) and upload it to `device`.  CK_EINVAL on malformed input (bad sizes, unbalanced
 * reaction when elem_comp is given, non-positive A or W); CK_EUNSUPPORTED for more than 3 distinct
 * species on one side of a reaction or more than 8 distinct t_mid values. */
int32_t ck_mech_load(const ck_mech_desc* desc, int32_t device, ck_mech** out);
int32_t ck_mech_free(ck_mech* m);

/* Kinetic model from CHEMKIN-II style text (ELEMENTS / SPECIES / THERMO with four-card NASA-7 entries / REACTIONS with
 * "<=>", "=", "=>", "+M", "(+M)", LOW/, TROE/, efficiencies, DUPLICATE; '!' comments; cm-mol-s-K, cal/mol): the
 * counterpart of the paper's `create_rate_subs` interpreter.  Host code, no device needed.  The
 * returned object owns the arrays ck_parsed_desc() points to; pass that description to ck_mech_load, then free it.
 * ck_parsed_name: species (what = 0) or element (what = 1) name number `index`.  CK_EINVAL with a line number in
 * ck_last_error() on malformed input. */
typedef struct ck_parsed ck_parsed;
int32_t ck_mech_parse(const char* text, ck_parsed** out);
const ck_mech_desc* ck_parsed_desc(const ck_parsed* p);
int32_t ck_parsed_name(const ck_parsed* p, int32_t what, int32_t index, char* buf, int32_t len);
int32_t ck_parsed_free(ck_parsed* p);
int32_t ck_mech_sizes(const ck_mech* m, int32_t* n_species, int32_t* n_reactions);
/* Reactor kind the handle's compute calls model (default CK_CONST_PRESSURE, Eq. 12-13).  CK_CONST_VOLUME (PAPER.md:107:
 * "a constant-volume process, i.e., where rho is constant, can be modeled by replacing c_p with c_v and h_k with u_k in
 * Eq. (13)"): the mass density of each reactor is fixed and the `p` argument of ck_rhs / ck_jac* / ck_integrate_* then
 * holds that density rho[n] in g/cm^3 instead of the pressure (the pressure follows from p = rho R_u T sum_k Y_k/W_k).
 * Not thread-safe against compute calls running on the same handle; load a second handle to use both kinds at once. */
int32_t ck_mech_set_reactor(ck_mech* m, int32_t kind);

/* Scratch bytes ck_integrate_{ros,rkf45} / ck_jac_batched need for n reactors (op = CK_OP_*). */
int32_t ck_workspace_bytes(const ck_mech* m, int32_t op, int64_t n, size_t* bytes);

/* dydt = f(y; p): Eq. 12-19.  y[(K+1) x ld], p[n], dydt[(K+1) x ld_out]. n = 0 is a no-op. */
int32_t ck_rhs(const ck_mech* m, int64_t n, const double* y, int64_t ld, const double* p, double* dydt,
               int64_t ld_out, void* stream);

/* J[(i*N + j)*ldJ + r] = d f_i / d y_j at constant p (dense N x N, all K species kept).
 * mode CK_JAC_ANALYTIC: hand-derived derivatives of Eq. 12-19.  mode CK_JAC_FD: first-order forward
 * differences with the CVODE-style increment (h, rtol, atol enter the increment only). */
int32_t ck_jac(const ck_mech* m, int64_t n, const double* y, int64_t ld, const double* p, int32_t mode, double h,
               double rtol, double atol, double* J, int64_t ldJ, void* stream);

/* The analytic Jacobian of ck_jac evaluated thread-per-reactor for large batches (one reactor per lane, one matrix
 * row at a time in tensor memory): same output layout as ck_jac.  Needs
 * ck_workspace_bytes(m, CK_OP_JAC, n) bytes of scratch; CK_EUNSUPPORTED for models with more than 123 species. */
int32_t ck_jac_batched(const ck_mech* m, int64_t n, const double* y, int64_t ld, const double* p, double* J, int64_t ldJ,
                       void* ws, size_t ws_bytes, void* stream);

/* ck_jac_batched for callers that cannot allocate (CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): same kernels, same output, but the scratch lives in a file-scope device array of CK_JAC_STATIC_BYTES that
 * every GPU loading the library holds until exit (the driver maps it with the module, lazily: on the first use of this
 * entry point on that device) -- no workspace argument, no cudaMalloc / cudaFree inside.
 * CK_EWORKSPACE (with the limit in ck_last_error()) when n reactors of this model need more scratch than that;
 * ck_jac_static_max_reactors gives the largest n that fits (2,761 for a 53-species / 325-reaction model, 1,161 for
 * 111 / 784).  All calls on one device share the array, which keeps the last call's contents (nothing needs clearing:
 * every entry is written before it is read): calls that OVERLAP on the GPU race -- serialise them on one stream. */
#define CK_JAC_STATIC_BYTES (32u << 20)
int32_t ck_jac_batched_static(const ck_mech* m, int64_t n, const double* y, int64_t ld, const double* p, double* J,
                              int64_t ldJ, void* stream);
int32_t ck_jac_static_max_reactors(const ck_mech* m, int64_t* n_max);

/* The per-reactor dense linear algebra of the Rosenbrock stage equations on its own (Eq. 6; cost
 * ~ N^3): for each of n systems factor A_r (row-major N x N at A + r N N, not modified) with partial
 * pivoting (first maximal |a| wins ties) and solve A_r x_r = b_r (b, x: [n][N]).  status[r] (optional) = CK_ST_OK or
 * CK_ST_ZERO_PIVOT.  Device pointers; 1 <= N <= 128.  One warp per system, blocked right-looking LU whose trailing
 * update runs on the FP64 tensor cores (mma.sync.m8n8k4.f64). */
int32_t ck_lu_solve_batched(int32_t N, int64_t n, const double* A, const double* b, double* x, int32_t* status, void* stream);

/* Advance every reactor from t = 0 to t = dt in place with the 4-stage Rosenbrock method ROS4
 * (Eq. 6-7, Table C.3) resp. the embedded Runge-Kutta-Fehlberg 4(5) pair (Eq. 2-3,
 * PAPER.md:49-63, Table B.2) under adaptive step-size control (Algorithm 1/2).
 * n_accept / n_reject / status / h_last are per-reactor device arrays [n] (each may be NULL).
 * A failed reactor keeps its last accepted state; the call still returns CK_OK.
 * ws must hold ck_workspace_bytes(...) bytes, else CK_EWORKSPACE. */
int32_t ck_integrate_ros(const ck_mech* m, int64_t n, double* y_inout, int64_t ld, const double* p, double dt,
                         const ck_opts* opts, int32_t* n_accept, int32_t* n_reject, int32_t* status, double* h_last,
                         void* ws, size_t ws_bytes, ck_report* report, void* stream);
int32_t ck_integrate_rkf45(const ck_mech* m, int64_t n, double* y_inout, int64_t ld, const double* p, double dt,
                           const ck_opts* opts, int32_t* n_accept, int32_t* n_reject, int32_t* status,
                           double* h_last, void* ws, size_t ws_bytes, ck_report* report, void* stream);

/* HOST-buffer variants (end-to-end path): same semantics, all batch pointers are host pointers; the
 * library stages them through device buffers it allocates (and caches in the handle), including the
 * workspace, and synchronises before returning. */
int32_t ck_rhs_host(ck_mech* m, int64_t n, const double* y, int64_t ld, const double* p, double* dydt, int64_t ld_out);
int32_t ck_integrate_host(ck_mech* m, int32_t op, int64_t n, double* y_inout, int64_t ld, const double* p, double dt,
                          const ck_opts* opts, int32_t* n_accept, int32_t* n_reject, int32_t* status, double* h_last,
                          ck_report* report);

/* Roofline support: FP64 instruction count ("slots": DFMA/DMUL/DADD, transcendental at their FP64-pipe
 * instruction counts) that one RHS evaluation of this mechanism needs algorithmically. */
int32_t ck_rhs_slots(const ck_mech* m, double* slots);
/* Which kernel ck_rhs launches for n states of this model: threads per CTA and whether the production-rate
 * accumulators live in tensor memory (rhs_kernel_tmem<block>) or in shared memory (rhs_kernel<block>). */
int32_t ck_rhs_variant(const ck_mech* m, int64_t n, int32_t* block, int32_t* tmem);
/* Measure the FP64 FMA peak of the device with a register-resident DFMA chain (slots/s). */
int32_t ck_fp64_peak(int32_t device, double* dfma_per_s, void* stream);
/* The same through the FP64 tensor cores (mma.sync.m8n8k4.f64, 256 FMA per warp instruction): FMA/s.  On B200 it equals
 * the vector rate (64 FMA/clk/SM), so DMMA buys instruction count and operand traffic, not flops. */
int32_t ck_fp64_mma_peak(int32_t device, double* fma_per_s, void* stream);

/* Waste of each SIMD work unit, Eq. 20: W_j = 1 - sum_i N_i / (P max_i N_i) over the P
 * consecutive reactors of unit j under the static linear reactor -> lane mapping, N_i = attempts of
 * reactor i = n_accept[i] + n_reject[i] (n_reject may be null).  All pointers are device pointers owned by the
 * caller; W has ceil(n / P) entries.  The ragged last unit divides by the lanes it has; a unit whose reactors took
 * no step has W = 0.  P in [1, 1024].  Enqueues on `stream`. */
int32_t ck_waste(int64_t n, const int32_t* n_accept, const int32_t* n_reject, int32_t P, double* W, void* stream);
/* The same metric when every lane works through `tasks` reactors instead of one (the mitigation of Murray's ref. [48],
 * PAPER.md:419): unit j holds P x tasks consecutive reactors, lane l takes reactors l, l + P, l + 2 P, ... of the unit,
 * its cost is the sum of their attempts, W_j = 1 - sum_i N_i / (lanes x max_l cost_l), lanes = lanes that own at least
 * one reactor.  W has ceil(n / (P tasks)) entries; tasks = 1 is ck_waste.  1 <= tasks <= 4096. */
int32_t ck_waste_tasks(int64_t n, const int32_t* n_accept, const int32_t* n_reject, int32_t P, int32_t tasks, double* W,
                       void* stream);

#ifdef __cplusplus
}
#endif
#endif /* CK_H_ */
