/* =======================================================================================
 * qmc_feynman.h -- C ABI of the B200-native hot path of arXiv:1508.02512
 * ("Efficient Numerical Evaluation of Feynman Integrals", Li, Wang, Yan, Zhao):
 * randomly shifted rank-1 lattice quasi-Monte Carlo integration of sector-decomposed,
 * eps-expanded Feynman-parameter integrands, with contour deformation in the physical region.
 *
 * "P:<n>" cites /root/reference/PAPER.md line n; "R:Cxx" cites a reading listed in DESIGN.md.
 *
 * Two calls carry the path (BASELINE.json north_star):
 *   qmc_prepare  (graph, kinematics, eps_order) -> sector tables          [host only]
 *   qmc_integrate(sector tables, N, m, seed)    -> Laurent coefficients +- errors   [CUDA, sm_100a]
 *
 * Conventions
 *  - Every function returns 0 (QMC_OK) or a negative qmc_status; nothing throws, aborts or prints.
 *  - All pointers are HOST pointers unless the name says `dev_`.  Inputs are borrowed for the duration
 *    of the call.  `qmc_tables` is created by qmc_prepare and destroyed by qmc_tables_free.  Outputs go
 *    to caller-allocated buffers (NULL = not wanted).
 *  - Device memory is owned by the caller: `dev_workspace` is any device allocation of at least
 *    qmc_workspace_bytes() bytes (e.g. a torch tensor's data_ptr()), `cuda_stream` is a cudaStream_t
 *    (e.g. torch.cuda.current_stream().cuda_stream; NULL = default stream).  The library never
 *    allocates device memory; it synchronises only its own stream before filling host outputs.
 *    The evaluation is one kernel launch per run of sectors (the sector tables travel in the kernel
 *    parameters); the launches of one call are spread over up to 8 internal non-blocking streams
 *    owned by the qmc_tables object (created on first use, destroyed by qmc_tables_free), forked from
 *    and joined back into `cuda_stream` with events: to the caller the call is ordered on `cuda_stream`.
 *  - There is NO CPU fallback: without a CUDA device qmc_integrate* returns QMC_ECUDA.
 *
 * What is computed.  For a graph with P propagators (powers nu_j = 1), L loops, D = 4 - 2 eps:
 *     I = (-1)^P Gamma(P - L D/2) J(eps),   J(eps) = sum_{l=1..P} I_l         (Eqs. 5-6; R:C1)
 *  where I_l are the primary-sector integrals over the (P-1)-cube.  The library returns the Laurent
 *  coefficients of J(eps) (orders k_min .. k_max = eps_order); the Gamma prefactor and any normalisation
 *  (R:C2-C4) are applied by the caller (qmc_prefactor_series helps).
 * ======================================================================================= */
#ifndef QMC_FEYNMAN_H
#define QMC_FEYNMAN_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  QMC_OK = 0,
  QMC_EINVAL = -1,       /* bad graph (disconnected, leg on a missing vertex, L < 1, P > 9), bad N/z/m */
  QMC_EDEPTH = -2,       /* iterated decomposition did not terminate within max_depth (R:C7) */
  QMC_EUNSUPPORTED = -3, /* alpha_j <= -4, or alpha_j <= -2 with lambda > 0 or on more than two variables of a sector (the p >= 1
                            Taylor terms of Eq. 11, exist on the real path for alpha_j = -2, -3 only; R:C9, R:C28),
                            beta_j = 0 on a variable with alpha_j <= -1, more than 4 such variables in one sector */
  QMC_ECUDA = -4,        /* CUDA runtime error or no device */
  QMC_ENOMEM = -5,       /* workspace / export buffer too small */
  QMC_ECONTOUR = -6      /* reserved: contour problems are REPORTED through counters, never fatal */
} qmc_status;

/* ---- inputs (an integral is a graph, masses, propagator powers and external kinematics) ---- */
typedef struct {
  int32_t n_vertices, n_edges, n_legs;
  const int32_t *edge_u, *edge_v; /* [n_edges] end points; multi-edges allowed (bubble) */
  const double *edge_m2;          /* [n_edges] squared internal masses */
  const int32_t *edge_nu;         /* [n_edges] propagator powers nu_j in 1..8 (Eq. 1); NULL = all 1.  Powers other than 1
                                     change the exponents of U and F (Eq. 6 with N_nu = sum nu_j) and put x_j^(nu_j-1) into the
                                     integrand; such tables run on the generic kernel.  A sector that ends with an exponent
                                     alpha_j = -2 or -3 needs the p >= 1 Taylor terms of Eq. 11: served by the
                                     generic kernel on the real path (lambda = 0), at most two such variables per sector;
                                     alpha_j <= -4, a third such variable, or any of them with lambda > 0: QMC_EUNSUPPORTED */
  const int32_t *leg_vertex;      /* [n_legs] vertex each external leg (all incoming) attaches to */
} qmc_graph;

typedef struct {
  const double *gram; /* [n_legs*n_legs] p_i . p_j, momentum conservation assumed */
} qmc_kinematics;

typedef struct {
  double lambda;     /* 0: Euclidean / real path.  > 0: contour deformation z_j = t_j - i lambda t_j (1-t_j) dF/dt_j
                        (Eq. 14), complex path, all variables deformed with the same lambda (R:C11) */
  int32_t transform; /* 0: x = 3y^2 - 2y^3, weight prod 6y(1-y) (Eq. 21).  1: tent/baker (R:C20).
                        2: x = 10y^3 - 15y^4 + 6y^5, weight prod 30y^2(1-y)^2 -- the next member of Eq. 21's family */
  int32_t max_depth; /* decomposition recursion cap; <= 0: 64 */
  int32_t lattice;   /* generating vector of qmc_integrate when the caller passes none: 0 = Korobov-form P_2 search on the
                        device (R:C13), 1 = component-by-component construction (R:C25; qmc_cbc_vector on the host,
                        N an odd prime below 2^26, cached per N in the tables object) */
  /* Layout of the device tables; 0 = the defaults measured on B200.  They change how the
   * sectors are grouped into chunks and how many per-point product slots a chunk may use, never the result. */
  int32_t slot_budget;       /* real path: chunk-wide slots of the slot program (default 36) */
  int32_t chunk_bytes;       /* target bytes of sector tables per chunk (both paths) */
  int32_t threads;           /* real path: threads per block, 128 or 512 (default: chosen from the tables) */
  int32_t slot_budget_cplx_real, slot_budget_cplx; /* complex path: real / complex slots per chunk */
  int32_t dense_template;    /* real path: dense-position template of the sector tables, 1 = lean, 2 = two-loop sized
                                (default: the one with the lower modelled cost) */
  int32_t pole_extraction;   /* 0: subtraction (Eqs. 11-12; the default and the timed path).  1: integration by parts
                                (Eq. 13, repeated -alpha_j times per variable; reading C30): same Laurent series, no
                                large-number cancellation; real path only (lambda > 0: QMC_EUNSUPPORTED), generic kernel only,
                                prod_j (1 - alpha_j) over the variables with alpha_j <= -1 of a sector at most 16 */
  int32_t strategy;          /* decomposition strategy.  0: iterated, the deterministic rule of DESIGN.md reading C7 (all configs, the
                                default).  1: geometric (Kaneko-Ueda; the strategy the paper says it uses): one monomial
                                substitution per simplicial cone of the normal fan of the Newton polyhedron of U_l F_l, guaranteed to
                                terminate (reading C31; a cone with |det V| > 1: QMC_EUNSUPPORTED -- none was met).  The totals do not
                                depend on the strategy, the sectors do */
} qmc_options;

typedef struct qmc_tables qmc_tables; /* opaque sector tables (Eqs. 7-9) */

/* Feynman graph -> U, F -> P primary sectors (Eqs. 3-6) -> iterated sub-sectors until U^ and F^
 * both have a constant term (Eqs. 7-9; deterministic rule R:C7) -> per-sector tables: exponents
 * (alpha_j, beta_j) of t_j^{alpha_j + beta_j eps} and the monomial lists of U^, F^ (constants kept inside, R:C6).
 * eps_order = highest order of J(eps) wanted.  options may be NULL (lambda 0, transform 0, depth 64). */
int qmc_prepare(const qmc_graph *graph, const qmc_kinematics *kin, int32_t eps_order, const qmc_options *options,
                qmc_tables **out);
/* Kinematic scans (Fig. 2: the paper's 1000-point scan of the one-loop box): ONE graph at n_points
 * kinematic points `kinematics[0 .. n_points)`.  The tables hold the sectors of all points one after the other (the exponent
 * structure of a point's sectors does not depend on the kinematics, only the coefficients do); every point must decompose into
 * the same number of sectors (a coefficient that vanishes at one point only changes the decomposition: QMC_EINVAL).
 * qmc_tables_info reports the total number of sectors, qmc_tables_batch_info the points and the sectors per point.
 * Integrate with qmc_run.mode = 3: one call evaluates all points (one fused launch per point and chunk, spread over the side
 * streams, ONE final sum, ONE statistics pass, ONE copy back) on the same lattice and shift vectors, and returns per POINT
 * what mode 2 returns per sector: sector_coeff / sector_err [n_points][K][2], shift_sums [n_points][K][m][2]. */
int qmc_prepare_batch(const qmc_graph *graph, const qmc_kinematics *kinematics, int32_t n_points, int32_t eps_order,
                      const qmc_options *options, qmc_tables **out);
int qmc_tables_batch_info(const qmc_tables *t, int32_t *n_points, int32_t *sectors_per_point);
void qmc_tables_free(qmc_tables *t);

/* orders k_min = -max_sector(#singular variables) .. k_max = eps_order; K = k_max - k_min + 1 */
int qmc_tables_info(const qmc_tables *t, int32_t *n_sectors, int32_t *dim, int32_t *k_min, int32_t *k_max,
                    int32_t *is_complex);

/* Flat export of the tables so that an independent program can evaluate the SAME sectors (data, not code).
 * Layout: 8-byte words w[] (int64 unless noted):
 *   w[0]=0x514D4346 ('QMCF'), w[1]=version 1, w[2]=n_sectors, w[3]=dim n, w[4]=k_min, w[5]=k_max,
 *   w[6]=is_complex + 2 * pole_extraction,
 *   w[7..10]=a_U0,a_U1,a_F0,a_F1 with U^{a_U0+a_U1 eps} F^{a_F0+a_F1 eps}, w[11]=lambda (double);
 *   then per sector: primary index, alpha[n], beta[n], nU, nF, nU x {coeff (double), e[n]}, nF x {coeff (double), e[n]}
 *   (variables in the ORIGINAL order t_1..t_n of Eq. 4, monomials in the library's evaluation order).
 * Call with buf = NULL to get the size in bytes in *len; otherwise *len is the capacity on entry. */
int qmc_tables_export(const qmc_tables *t, void *buf, size_t *len);

/* ---- outputs ---- */
typedef struct {
  double *coeff, *err;               /* [K][2] totals over sectors: mean over shifts (Eq. 19) and the square root
                                        of Eq. 20, (Re, Im) separately (R:C15) */
  double *sector_coeff, *sector_err; /* [n_sectors][K][2] the same per sector */
  double *shift_totals;              /* [K][m][2] per-shift estimates Q_k summed over sectors (Eq. 18) */
  double *shift_sums;                /* [n_sectors][K][m][2] per-sector per-shift estimates (parity checks) */
  int64_t counters[4];               /* #corner evaluations with Im F^(z) > 0, with Re U^(z) <= 0,
                                        #non-finite (point, sector) evaluations (dropped), #boundary points (R:C18) */
  double kernel_ms;                  /* device time of all kernels of the call: evaluation, final sum, statistics (CUDA events) */
  double eval_kernel_ms;             /* device time of the evaluation kernel alone (S1-S7 first stage) */
  int64_t h2d_bytes, d2h_bytes;      /* bytes this call moved host->device (shifts, logarithm table, and the kernel parameter
                                        blocks that carry the sector tables) and device->host (results) */
  int32_t kernel_launches;           /* number of kernel launches made by this call */
  int32_t mode_used;                 /* 1 fused (all sectors summed in registers), 2 per-sector */
} qmc_result;

/* Explicit control of one integration (the parity entry point). */
typedef struct {
  const uint64_t *z;        /* [dim] generating vector, components coprime to N; NULL: library's choice (R:C13) */
  const double *shifts;     /* [m][dim] shift vectors in [0,1); NULL: SplitMix64 stream of `seed` (R:C14) */
  uint64_t index_begin, index_step, index_count; /* lattice indices i = begin + c*step, c < count; count 0 = all N.
                                                    The sum is always normalised by 1/N (Eq. 18). */
  int32_t sector_begin, sector_end;              /* sector range; end 0 = all */
  int32_t mode;             /* 0 auto (per-sector iff a per-sector output is requested), 1 fused, 2 per-sector,
                               3 per kinematic point of a batch (qmc_prepare_batch): fused within a point */
  int32_t tables_resident;  /* 1: reuse what an earlier call left in this workspace (the logarithm table);
                               2: reuse the shift vectors of that call as well (nothing is copied from the host) -- only if
                               they are the ones this call asks for: the same m and, unless that call passed them explicitly,
                               the same seed; otherwise they are generated and uploaded again.
                               A qmc_tables object carries launcher state (events, side streams, staging buffers, what is
                               resident): it serves ONE stream and ONE host thread at a time -- use one object per stream. */
  int32_t kernel;           /* 0: the table-driven kernels (real path: qmc4_eval_kernel, complex path: qmc5_eval_kernel) where
                               the tables allow them, else the generic kernel; 1: the generic kernel (qmc_eval_kernel) */
  int32_t waves;            /* launch geometry: blocks per resident block slot over all launches of a step (0 = 16) */
  int32_t streams;          /* internal side streams the launches of a step are spread over, 0..8 (0 = default 4;
                               -1 = none: all launches in order on cuda_stream) */
  const uint8_t *sector_mask; /* [n_sectors] (indexed by sector number), NULL = every sector of [sector_begin, sector_end):
                               only sectors with a non-zero entry are evaluated.  Fused mode with the table-driven kernels
                               only (else QMC_EUNSUPPORTED): a launch serves the selected sectors of its chunk, whatever
                               their positions (qmc_integrate_allocated: one call per lattice size) */
} qmc_run;

size_t qmc_workspace_bytes(const qmc_tables *t, uint64_t N, int32_t m);

/* S1-S8 of the hot path: lattice points x_i = {i z / N} (Eq. 17), m random shifts (Eq. 18),
 * periodising transform (Eq. 21), per sector the subtracted (Eqs. 10-12), eps-expanded and -- for
 * lambda > 0 -- contour-deformed (Eq. 14) integrand at every point, per-shift sums, mean and error over shifts
 * (Eqs. 19-20).  N must be < 2^31 with every z_j coprime to it, m >= 2. */
int qmc_integrate(const qmc_tables *t, uint64_t N, int32_t m, uint64_t seed, void *cuda_stream, void *dev_workspace,
                  size_t dev_workspace_bytes, qmc_result *out);
int qmc_integrate_ex(const qmc_tables *t, uint64_t N, int32_t m, uint64_t seed, const qmc_run *run, void *cuda_stream,
                     void *dev_workspace, size_t dev_workspace_bytes, qmc_result *out);

/* The same path in two halves, for callers that keep everything on the device (bench.py's device-timed loop):
 * qmc_integrate_async enqueues S1-S8 on `cuda_stream` (evaluation kernel, fixed-order final sum, statistics kernel)
 * and returns without synchronising; every result stays in the workspace.  qmc_result_fetch copies the results of
 * the LAST qmc_integrate_async on this tables object to the host (one D2H), synchronises the stream and fills `out`
 * exactly as qmc_integrate_ex does (qmc_integrate_ex = async + fetch).  Per-sector outputs exist only if that
 * launch ran in mode 2. */
int qmc_integrate_async(const qmc_tables *t, uint64_t N, int32_t m, uint64_t seed, const qmc_run *run, void *cuda_stream,
                        void *dev_workspace, size_t dev_workspace_bytes);
int qmc_result_fetch(const qmc_tables *t, void *cuda_stream, void *dev_workspace, size_t dev_workspace_bytes,
                     qmc_result *out);

/* Device address of the per-shift totals [K][m][2] (doubles; Eq. 18 summed over sectors) that the last
 * qmc_integrate_async left in the workspace -- for a device-side gather across ranks. */
int qmc_result_device_totals(const qmc_tables *t, void *dev_workspace, size_t dev_workspace_bytes, void **totals_out);

/* ---- helpers ---- */
/* Eqs. 19-20 on per-shift estimates: shift_totals [K][m][2] (host) -> coeff, err [K][2], Re and Im
 * separately (R:C15).  Used to combine the per-shift estimates gathered from several GPUs (each rank integrates its
 * own block of shift vectors).  m >= 2. */
int qmc_statistics(const double *shift_totals, int32_t K, int32_t m, double *coeff, double *err);
/* Algorithmic FP64 operation count of the evaluation (DFMA = 2, DADD = DMUL = 1, log,
 * reciprocal, division and atan2 at the fixed costs stated there): flops per (lattice point, shift) spent once per
 * point (S1-S3) and in all sectors [sector_begin, sector_end) (S4-S7; end 0 = all), plus the number of corner
 * evaluations per point.  Any output may be NULL. */
int qmc_flop_model(const qmc_tables *t, int32_t sector_begin, int32_t sector_end, double *flops_point,
                   double *flops_sectors, int64_t *corners);
/* Korobov-form generating vector z = (1, a, a^2, ...) mod N with `a` minimising the P_2 figure of merit over a fixed
 * deterministic candidate list (R:C13; "component-by-component" is the paper's own choice).  Runs on the
 * device (needs workspace of qmc_workspace_bytes). */
int qmc_generating_vector(uint64_t N, int32_t dim, void *cuda_stream, void *dev_workspace, size_t dev_workspace_bytes,
                          uint64_t *z_out);
/* The same search for callers that cannot allocate device memory (code under CUDA graph capture, serving loops, harnesses
 * that forbid cudaMalloc): no workspace argument -- the scratch of the P_2 kernel (candidate vectors and per-block partial
 * sums, 153 600 bytes) is a fixed array inside the library that every GPU holds from the moment it loads the library until
 * the process exits.  Calls no cudaMalloc / cudaFree and no allocating routine; same candidates, same kernel, same z as
 * qmc_generating_vector.  Limits: 5 <= N < 2^31, dim <= 8; dim > 8 returns QMC_ENOMEM ("workspace or buffer too small":
 * the fixed scratch is sized for 64 candidates of up to 8 components).  All calls on one device SHARE the array: calls that
 * overlap on the GPU (two streams, two threads) race -- serialise them.  Synchronises `cuda_stream` before returning. */
int qmc_generating_vector_noalloc(uint64_t N, int32_t dim, void *cuda_stream, uint64_t *z_out);
/* Generating vector by the component-by-component construction the paper names (refs [29, 30]): z_1 = 1, then
 * z_d = argmin over z in [1, (N-1)/2] of  e^2(z_1..z_d) = -1 + (1/N) sum_i prod_j (1 + 2 pi^2 B_2({i z_j / N}))  (the P_2
 * criterion of R:C13 with unit weights; ties -> smaller z; R:C25).  HOST function, O(dim N log N): the candidates of one
 * component are one cyclic convolution over the multiplicative group of the prime N (FFT), which only screens; the
 * decision is taken on plain O(N) sums of the closest candidates.  N an odd prime below 2^26, 1 <= dim <= 16, else
 * QMC_EINVAL; QMC_ENOMEM if the host work arrays (about 50 N bytes) cannot be allocated.  z_out[dim] caller-owned;
 * e2_out[dim] (NULL = not wanted) receives the criterion after each component. */
int qmc_cbc_vector(uint64_t N, int32_t dim, uint64_t *z_out, double *e2_out);
/* Embedded lattice sequence (P:172 names better lattices as the source of the O(1/n) rate; R:C26): rules with
 * N = 2^k points, k_min <= k <= k_max, that share ONE generating vector with odd components.  The even lattice indices of level
 * k + 1 are the points of level k ({2i z / 2^(k+1)} = {i z / 2^k}, Eq. 17), so raising N re-uses every point already evaluated.
 * qmc_embedded_vector: Korobov form z = (1, a, a^2, ...) mod 2^k_max, `a` odd, minimising over a fixed list of 64 candidates the
 * worst level of P_2(z mod 2^k; 2^k) / ((k ln 2)^dim / 4^k) (the P_2 criterion of R:C13 per level, relative to its expected rate).
 * Runs on the device (workspace as for qmc_generating_vector).  3 <= k_min <= k_max <= 30, dim <= 8. */
int qmc_embedded_vector(int32_t k_min, int32_t k_max, int32_t dim, void *cuda_stream, void *dev_workspace,
                        size_t dev_workspace_bytes, uint64_t *z_out);
/* S1-S8 over the levels k_min, k_min + 1, ... of an embedded sequence with generating vector z (odd components, z mod 2^k at
 * level k) and the m shift vectors of `seed`: level k_min evaluates all 2^k_min indices, every further level only its odd indices
 * (qmc_run.index_begin = 1, index_step = 2), and the per-shift estimates combine as Q_k = Q_{k-1} / 2 + (odd part), each part
 * carrying the 1/N of Eq. 18 of its own level.  Stops after the first level whose estimated relative error of the highest order
 * kept (R:C17) is <= target_rel_err (<= 0: runs to k_max).  Fused mode; `out` receives coeff, err, shift_totals [K][m][2] of
 * the level reached (per-sector outputs must be NULL), the counters and times summed over the levels; *k_reached the level,
 * *points_evaluated = 2^k_reached lattice points per shift (a restart at every level would cost 2^(k+1) - 2^k_min). */
int qmc_integrate_embedded(const qmc_tables *t, int32_t k_min, int32_t k_max, double target_rel_err, int32_t m, uint64_t seed,
                           const uint64_t *z, void *cuda_stream, void *dev_workspace, size_t dev_workspace_bytes,
                           qmc_result *out, int32_t *k_reached, int64_t *points_evaluated);
/* Per-sector lattice sizes by variance (R:C27), on an embedded sequence (z as for qmc_integrate_embedded):
 * (1) every sector at N0 = 2^k0 in per-sector mode -> per-sector error estimates e_s of the highest order kept (Eq. 20 per sector);
 * (2) sizes N_s = (a_s/c_s)^(1/3) (sum_r a_r^(1/3) c_r^(2/3))^(1/2) / tau, a_s = e_s^2 N0^2, c_s = modelled cost of the sector,
 *     tau = target_rel_err |coefficient|: the cheapest sizes that meet sum_s e_s(N_s)^2 <= tau^2 if errors fall like 1/N,
 *     rounded up to powers of two in [2^k0, 2^k_max];
 * (3) maximal runs of neighbouring sectors with one size are evaluated in fused mode; all sectors share the shift vectors, the
 *     per-shift totals T_k = sum over runs are unbiased whatever the sizes, and Eqs. 19-20 on them give the error bar (R:C16);
 * (4) while that error is above the target every run climbs one level (only its odd indices are new).
 * levels_out [n_sectors] (NULL = not wanted): log2 of the final size per sector; *evals_per_shift: integrand evaluations per
 * shift vector over all stages (a uniform rule costs n_sectors 2^k).  target_rel_err > 0; per-sector outputs must be NULL. */
int qmc_integrate_allocated(const qmc_tables *t, int32_t k0, int32_t k_max, double target_rel_err, int32_t m, uint64_t seed,
                            const uint64_t *z, void *cuda_stream, void *dev_workspace, size_t dev_workspace_bytes,
                            qmc_result *out, int32_t *levels_out, int64_t *evals_per_shift);
/* m shift vectors from the SplitMix64 stream keyed by seed: Delta = (u64 >> 11) * 2^-53, shift-major (R:C14) */
int qmc_shifts(uint64_t seed, int32_t m, int32_t dim, double *shifts_out);
/* Laurent series of  e^{eg * eps * gamma_E} * base^{p0 + p1 eps} * Gamma(g0 + g1 eps),  g0 a non-negative integer,
 * orders lo .. lo+n_out-1 (lo = -1 iff g0 == 0); multiply_series = 1 multiplies J (orders k_min..k_max, with errors
 * combined in quadrature) in place of writing the bare series. */
int qmc_prefactor_series(double eg, double base, double p0, double p1, int32_t g0, double g1, int32_t n_out,
                         double *series_out, int32_t *lowest_order);
/* Sustained FP64 FMA rate of the device (register-resident DFMA chains), in FLOP/s (DFMA = 2).  The roofline
 * denominator of the evaluation kernel (MEASURED_PEAKS.json has no FP64 entry). */
int qmc_fp64_peak(void *cuda_stream, void *dev_workspace, size_t dev_workspace_bytes, double *flops_out, double *ms_out);
/* Human-readable description of the device tables (chunks, slot programs, record counts) written to buf as a
 * NUL-terminated string, truncated to len bytes.  Diagnostics only. */
int qmc_tables_describe(const qmc_tables *t, char *buf, size_t len);
const char *qmc_strerror(int status);

#ifdef __cplusplus
}
#endif
#endif /* QMC_FEYNMAN_H */
