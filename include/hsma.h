/*
 * hsma.h -- C-ABI of the B200-native hot path of the harmonic surface mapping algorithm
 * (HSMA, arXiv 1806.04801).  Citations are PAPER.md line numbers;
 * "reading Sx/Gx" refers to DESIGN.md "Readings of the paper".
 *
 * The library computes, entirely in CUDA kernels for sm_100a (there is no CPU fallback):
 *   (a) Phi_in at the monitoring (check) points, summed over the near image cells   Eq.(5)
 *   (-) the least-squares fit of the harmonic coefficients A_nm                     Eq.(7)
 *   (-) the harmonic surface mapping A_nm -> surface charge + dipole per node       Eq.(10),(11) PAPER.md:99-105
 *   (b) Phi_in at all N sources over the near image cells, self excluded
 *   (c) Phi_out at all N sources from the M sphere nodes (charge + dipole)          Eq.(10), Eq.(16)
 *   (-) U = 1/2 sum q_i phi_i
 *
 * Conventions
 *   - every call returns an hsma_status; nothing throws or aborts; out-params are untouched on error.
 *   - "dev" pointers are CUDA device pointers owned by the caller; "host" pointers are host memory.
 *   - Gaussian units, G = 1/r (Eq.1).  Coordinates are box coordinates in [0, L_a];
 *     the library centres them (reading G10).
 *   - periodic kinds: phi is in the gauge A_00 = 0 (reading S2); U is gauge free for neutral input.
 *   - hsma_evaluate* are asynchronous on the plan's stream and perform no host synchronisation
 *     (hsma_evaluate_host synchronises because it returns host data; the first evaluate at a larger N than before grows
 *     the plan's scratch with cudaFree/cudaMalloc, an implicit device synchronisation -- see "Thread safety" below).
 *   - on a non-default stream, repeated evaluates with identical arguments (same pointers and sizes: the MD loop)
 *     are captured into one CUDA graph on the second call and replayed afterwards.
 *   - preconditions not checked: particles inside the box, no coincident particles, no particle on
 *     a check point (reading S13).
 */
#ifndef HSMA_H_
#define HSMA_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hsma_plan hsma_plan; /* opaque, library-owned */

typedef enum {
    HSMA_OK = 0,
    HSMA_ERR_INVALID_ARG = -1,
    HSMA_ERR_GEOMETRY = -2,       /* R_aux outside (R0, min_a (s_a+1/2) L_a]  (reading S7) */
    HSMA_ERR_NOT_NEUTRAL = -3,    /* periodic axes need sum q = 0             (reading S17) */
    HSMA_ERR_CUDA = -4,
    HSMA_ERR_ALLOC = -5,
    HSMA_ERR_RANK_DEFICIENT = -6, /* fitting matrix lost rank in the Householder QR */
    HSMA_ERR_TOO_LARGE = -7       /* hsma_direct_sum_static only: sizes beyond its fixed scratch */
} hsma_status;

typedef enum {
    HSMA_BC_PERIODIC = 0,                  /* Eq.(3): all axes periodic             */
    HSMA_BC_MIRROR_CAVITY = 1,             /* Eq.(4): all axes reflecting, gamma^|k| */
    HSMA_BC_SLAB_XY_PERIODIC_Z_MIRROR = 2  /* x,y periodic, z reflecting (readings G11, S16): with the far-data closure for
                                              any gamma; with the boundary closure for grounded plates, gamma = -1     */
} hsma_boundary_kind;

typedef enum {
    HSMA_CLOSURE_BOUNDARY = 0, /* residual of the boundary condition at the check points.  Periodic:
                                  K circumsphere points and their wrapped partners; cavity: K Dirichlet points on the
                                  faces; grounded slab: K circumsphere points wrapped in x,y only PLUS K Dirichlet points
                                  on the two plates (check_xyz, if given, are the plate points) -- DESIGN.md 6.8.
                                  On reflecting walls gamma must be -1 (conductor: Dirichlet rows Phi = 0) or +1
                                  (Neumann rows d Phi/d n = 0: wall points must lie exactly on a wall,
                                  the input must be neutral and phi is in the gauge A_00 = 0) */
    HSMA_CLOSURE_FAR_DATA = 1, /* rhs = direct sum over the far cell table (reading S16, config 4)       */
    HSMA_CLOSURE_FACE_PAIRS = 2 /* periodic kind only -- BASELINE.json's "check-point pairs on opposite faces" made
                                  well posed (reading S15): K points on the lower faces x_a = -L_a/2
                                  (check_xyz, or the library's lattice) and their partners on the opposite faces;
                                  each pair gives a value row AND a normal-derivative row (2K rows) */
} hsma_closure;

typedef enum {
    HSMA_QUAD_SPIRAL = 0, /* exactly M nodes, Hannay-Nye warp on a golden-angle spiral (reading S10) */
    HSMA_QUAD_LATTICE = 1 /* the paper's F1/F2 lattice, M = 2(F2+1), PAPER.md:124-126 (reading G4)   */
} hsma_quad_rule;

typedef enum {
    HSMA_NEAR_WHOLE_CELLS = 0, /* every image of the cells |k_a| <= near_shell[a], generated on the fly (reading S7) */
    HSMA_NEAR_SPHERE = 1       /* only the images inside the sphere |r| <= R_aux.  Each evaluate builds
                                  the explicit image list on the device (count, scan, scatter), packs it and sums it
                                  with the identity cell.  The length of the list never visits the host (buffers are
                                  sized for the whole cell table, the kernels read the count themselves): no host
                                  synchronisation, CUDA-graph replay as in the other modes.  A source outside the
                                  sphere is detected on the device and surfaces as HSMA_ERR_GEOMETRY at
                                  hsma_plan_sync.  Boundary closures only.  Ordered-pair kernels only: an image inside
                                  the sphere need not have its partner inside, so the symmetric form does not apply. */
} hsma_near_mode;

typedef enum {
    HSMA_NEAR_ALG_DIRECT = 0,  /* the exact direct sum over all pairs: near_sym_kernel / near_sum_kernel (north_star) */
    HSMA_NEAR_ALG_FMM = 1      /* SURVEY.md 8(f) NEXT 4, Table I: step (b) by a uniform-grid
                                  fast multipole method: O(N) instead of O(N^2), the same sum up to the
                                  truncation of the expansions (<= 1e-12 of max|phi| at the default order 20).  Used when an
                                  evaluate covers all N targets (potentials and forces; target shards and the multi-GPU
                                  phases keep the direct kernels); step (a) at the check targets is then served by the
                                  same multipoles (boundary closures without derivative rows).  Needs the whole-cell near set and box sides that are integer multiples of
                                  the smallest one (cubic FMM boxes): HSMA_ERR_INVALID_ARG at plan creation otherwise. */
    , HSMA_NEAR_ALG_AUTO = 2   /* the FMM from N = 36,864 sources on (the measured crossover is N ~ 35k) where the
                                  geometry allows it, the direct sum below and wherever the FMM does not apply; never an error */
} hsma_near_algorithm;

typedef enum {
    HSMA_DIPOLE_EXACT = 0,     /* exact normal dipole on the M nodes (reading S9) */
    HSMA_DIPOLE_FD3 = 1        /* Eq.(12)-(14) PAPER.md:107-120: central difference over three spheres, 3M charges */
} hsma_dipole_mode;

/* Plan descriptor (full form).  Set struct_size = sizeof(hsma_plan_desc); zero the rest first. */
typedef struct {
    size_t struct_size;
    int kind;             /* hsma_boundary_kind */
    double L[3];          /* box sides */
    int near_shell[3];    /* near cells |k_a| <= near_shell[a]; whole cells (reading S7) */
    double gamma;         /* reflection factor per mirror reflection (-1 = grounded metal; +1 = Neumann wall;
                             other values only with HSMA_CLOSURE_FAR_DATA) */
    double R_aux;         /* radius of the auxiliary sphere */
    int p;                /* harmonic degrees n = 0..p-1, p*p unknowns (reading S1); 1 <= p <= 32 */
    int M;                /* integration nodes on the sphere; M >= 8 */
    int K;                /* check points (periodic: K points + their K wrapped partners) */
    const double* check_xyz; /* host [K,3] CENTRED coordinates, or NULL: the library's rule
                                (periodic: Fibonacci grid on the circumsphere PAPER.md:82;
                                 otherwise a deterministic low-discrepancy set on the faces) */
    int closure;          /* hsma_closure */
    int far_shell[3];     /* HSMA_CLOSURE_FAR_DATA only: far table = cells within far_shell minus near */
    int quad_rule;        /* hsma_quad_rule */
    int rsqrt_refine;     /* refinement of the MUFU.RSQ64H seed in the source near sum (b):
                             1 = one mean-centred Newton step (|err| <= 1.2e-12 per pair, 10 FP64 instr/pair),
                             2 = one cubic (Halley) step (|err| <= 5e-16, 12 instr/pair),
                             0 = library default: 2 while N*N*cells < 2^32 pairs (latency-bound), else 1.
                             Steps (a) and (c) always use the cubic step. */
    /* paper-literal variants; 0 = the north_star forms */
    int near_mode;        /* hsma_near_mode */
    int dipole_mode;      /* hsma_dipole_mode */
    double fd_dr_rel;     /* HSMA_DIPOLE_FD3: Delta r / R_aux (1e-5; 1e-4 for the Dirichlet example); 0 = 1e-5 */
    /* sub-quadratic near sum; 0 = the direct sum */
    int near_algorithm;   /* hsma_near_algorithm */
    int fmm_order;        /* expansion order of the FMM, 2..30; 0 = 20 (truncation <= 1e-12 of max|phi|) */
    int fmm_levels;       /* leaf level of the FMM box hierarchy, 1..5; 0 = by N (about 500 sources per leaf) */
} hsma_plan_desc;

/*
 * north_star form: cubic box of side L, same shell on all axes, K = 2 p^2 check points (PAPER.md:163
 * N_m = 2P^2), gamma = -1 for mirror kinds, spiral nodes, boundary closure.
 * `cuda_stream` is a cudaStream_t (NULL = default stream); all work of the plan runs on it.
 * Preparation step of PAPER.md:140: cell table, check points, nodes, fitting matrix, its Householder
 * QR (device, single block).  Synchronises the stream before returning.
 */
hsma_status hsma_plan_create(double L, int boundary_kind, int near_shell, double R_aux, int p,
                             int M_fib, void* cuda_stream, hsma_plan** plan_out);
hsma_status hsma_plan_create_ex(const hsma_plan_desc* desc, void* cuda_stream, hsma_plan** plan_out);
hsma_status hsma_plan_destroy(hsma_plan* plan);

/*
 * Update step of PAPER.md:142 for N sources.
 *   xyz      dev [N,3] row-major box coordinates; q dev [N]
 *   phi_out  dev [N]   potential at every source (near images + sphere nodes, bare self term excluded)
 *   energy_out dev [1] U = 1/2 sum q_i phi_i, or NULL
 */
hsma_status hsma_evaluate(hsma_plan* plan, const double* xyz, const double* q, long long N,
                          double* phi_out, double* energy_out);
/*
 * Target-sharded form (multi-GPU): phi only at sources t0 <= i < t1;
 * phi_out dev [t1-t0]; energy_out dev [1] = 1/2 sum_{t0<=i<t1} q_i phi_i.  Step (a) and the fit are
 * computed in full (they need all sources).
 */
hsma_status hsma_evaluate_shard(hsma_plan* plan, const double* xyz, const double* q, long long N,
                                long long t0, long long t1, double* phi_out, double* energy_out);
/*
 * End-to-end form with HOST buffers: copies xyz,q to the device, evaluates, copies phi (and U) back,
 * synchronises.  phi_host [N] may be NULL (energy only); energy_host [1] may be NULL.
 */
hsma_status hsma_evaluate_host(hsma_plan* plan, const double* xyz_host, const double* q_host,
                               long long N, double* phi_host, double* energy_host);
/* Target-sharded end-to-end form: all N sources are copied in, phi_host [t1-t0] and the shard's
 * energy_host [1] are copied out.  hsma_evaluate_host is this with t0 = 0, t1 = N. */
hsma_status hsma_evaluate_shard_host(hsma_plan* plan, const double* xyz_host, const double* q_host,
                                     long long N, long long t0, long long t1, double* phi_host,
                                     double* energy_host);

/*
 * Forces (Eq.(9); Appendix A): as hsma_evaluate*, and in addition
 *   force_out dev [N,3] (shard: [t1-t0,3]) row-major,  F_i = -q_i grad [Phi_in + Phi_out](r_i),
 * with the bare self term excluded and the coefficients A_nm held fixed.  Steps (b) and (c) run their
 * potential+gradient kernels (16 / 26 FP64 instructions per pair instead of 10 / 17).  phi_out may be NULL.
 */
hsma_status hsma_evaluate_forces(hsma_plan* plan, const double* xyz, const double* q, long long N,
                                 double* phi_out, double* force_out, double* energy_out);
hsma_status hsma_evaluate_forces_shard(hsma_plan* plan, const double* xyz, const double* q, long long N,
                                       long long t0, long long t1, double* phi_out, double* force_out,
                                       double* energy_out);
/* HOST buffers; force_host [N,3] required, phi_host / energy_host may be NULL; synchronises. */
hsma_status hsma_evaluate_forces_host(hsma_plan* plan, const double* xyz_host, const double* q_host,
                                      long long N, double* phi_host, double* force_host, double* energy_host);

/*
 * Multi-GPU with step (a) sharded as well.  Every rank holds all N sources and the same plan.
 *   1. hsma_check_sums_shard      H1 + step (a) for the check targets c0 <= i < c1 (of K_t = plan_info[2]) only
 *   2. hsma_get_check_sums        copy that slice out: pc_out dev [c1-c0] (and pcg_out dev [c1-c0,3] when the fit has
 *                                 derivative rows -- Neumann walls, face-pair closure; else pcg_out may be NULL)
 *      ... the caller all-gathers the slices (K_t doubles: one latency-bound message) ...
 *   3. hsma_set_check_sums        copy the other ranks' slices in
 *   4. hsma_evaluate_rest_shard   H1 + fit + mapping + (b) + (c) + finish for the targets t0 <= i < t1 with the check
 *                                 sums as they now are; force_out may be NULL (potentials only)
 * All asynchronous on the plan's stream.  Steps 1 and 4 together equal hsma_evaluate(_forces)_shard.
 */
hsma_status hsma_check_sums_shard(hsma_plan* plan, const double* xyz, const double* q, long long N,
                                  long long c0, long long c1);
hsma_status hsma_get_check_sums(hsma_plan* plan, long long c0, long long c1, double* pc_out, double* pcg_out);
hsma_status hsma_set_check_sums(hsma_plan* plan, long long c0, long long c1, const double* pc_in, const double* pcg_in);
hsma_status hsma_evaluate_rest_shard(hsma_plan* plan, const double* xyz, const double* q, long long N,
                                     long long t0, long long t1, double* phi_out, double* force_out,
                                     double* energy_out);

/*
 * Step 4 in PART form: instead of a target shard, rank `part` of `n_parts` takes a contiguous
 * 1/n_parts of the UNORDERED source pairs of step (b) (symmetric form: one evaluation feeds phi_i and phi_j) and the
 * node sum (c) for the targets t0 <= i < t1 (the ranks' [t0,t1) must tile 0..N).  phi_part_out dev [N] (all targets),
 * force_part_out dev [N,3] (NULL: potentials only; with forces phi_part_out may be NULL) and energy_part_out dev [1]
 * (or NULL) are PARTIAL: their sums over the parts are phi, F and U -- the caller all-reduces them (2 MB / 6 MB at
 * N = 262,144).  Same arithmetic on every part count; results differ from the one-rank
 * evaluate only in the order of the sums.  Needs what the symmetric form needs: hsma_plan_part_form_applies(plan, N)
 * returns 1 if so (whole-cell near set, N > 7936, <= 128 near cells, pair form not forced to ordered), else 0 (use
 * hsma_evaluate_rest_shard);
 * HSMA_ERR_INVALID_ARG otherwise.
 */
hsma_status hsma_evaluate_rest_part(hsma_plan* plan, const double* xyz, const double* q, long long N, int part,
                                    int n_parts, long long t0, long long t1, double* phi_part_out,
                                    double* force_part_out, double* energy_part_out);
int hsma_plan_part_form_applies(const hsma_plan* plan, long long N);

/* Synchronise the plan's stream and return the sticky status of the evaluations since the last
 * call (HSMA_ERR_NOT_NEUTRAL, HSMA_ERR_CUDA, ...), then clear it. */
hsma_status hsma_plan_sync(hsma_plan* plan);

const char* hsma_status_string(int status);

/* ---- introspection / test and bench hooks ------------------------------------------------------- */
/* sizes: what[0]=rows of the fit, [1]=columns, [2]=check targets K_t, [3]=near cells, [4]=rhs cells,
 * [5]=M nodes, [6]=p, [7]=kernels launched by the last evaluate, [8]=near images summed per target by the last
 * evaluate (N * cells, or the image count inside the sphere), [9]=node records (M or 3M), [10]=1 if the fit has derivative rows (step (a) then also
 * produces grad Phi_in at the check targets), [11]=evaluates served by replaying the plan's CUDA graph.  host out [12]. */
hsma_status hsma_plan_info(hsma_plan* plan, long long* what_out);
/* copies of plan/evaluate state into caller DEVICE buffers (valid after an evaluate on the stream) */
hsma_status hsma_get_coeffs(hsma_plan* plan, double* A_out /* dev [p*p], R0-scaled basis */);
hsma_status hsma_get_rhs(hsma_plan* plan, double* rhs_out /* dev [rows] */);
hsma_status hsma_get_check_targets(hsma_plan* plan, double* xyz_out /* dev [K_t,3] centred */);
hsma_status hsma_get_nodes(hsma_plan* plan, double* xyz_out /* dev [M,3] */, double* w_out /* dev [M] */);
hsma_status hsma_get_surface(hsma_plan* plan, double* Q_out /* dev [M] */, double* P_out /* dev [M,3] dipole vectors */);
hsma_status hsma_get_fit_residual(hsma_plan* plan, double* rms_out /* host [1]; synchronises */);

/*
 * Raw kernel (a)/(b): phi[t] = sum_c w_c sum_j q_j / | tgt_t - (sign_c o src_j + shift_c) |  Eq.(5) PAPER.md:64.
 *   tgt dev [T,3], src dev [N,3] (both centred), q dev [N]; shift, sign HOST [C,3] (sign = +-1), w HOST [C].
 *   self_offset >= 0: target t is source self_offset+t, skipped in cell `central_cell` (-1: none).
 *   refine: 1 Newton / 2 cubic.  Runs on `cuda_stream`; synchronises it before returning (it frees its scratch).
 */
hsma_status hsma_direct_sum(const double* tgt, long long T, const double* src, const double* q,
                            long long N, const double* shift_host, const double* sign_host,
                            const double* w_host, int C, int central_cell, long long self_offset,
                            int refine, double* phi_out, void* cuda_stream);
/*
 * The same raw kernel for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): hsma_direct_sum_static calls no cudaMalloc / cudaFree / allocating library routine and
 * copies nothing from host memory (the cell table travels as a kernel argument).  All of its scratch -- cell table, packed
 * sources, slots, tile statistics, partial rows -- lives in ONE file-scope `static __device__` array of 16 MiB inside the
 * library (hsma_static_scratch_bytes), which every GPU that loads the library holds until the process exits.
 *   Arguments, layouts and result as hsma_direct_sum (Eq.(5)), with these limits: N <= 65,536 sources,
 *   T <= 65,536 targets, C <= 32 cells, and 16 MiB of scratch in all for the launch shape chosen (checked per call); beyond
 *   any of them the call returns HSMA_ERR_TOO_LARGE and launches nothing.  Other errors as hsma_direct_sum.
 *   Asynchronous: it enqueues 6 kernels on `cuda_stream` and returns without synchronising; phi_out is valid once the
 *   stream has passed them.  shift/sign/w are read before the call returns.
 *   EVERY call on a device shares the one array, which keeps the last call's contents (the call clears what must start at
 *   zero itself).  Calls on the same stream are ordered and safe; calls that can overlap on the GPU (different streams,
 *   different host threads; another process has its own copy) RACE on the scratch: serialise them.
 * hsma_static_scratch_setup: looks up the array's device address for the CURRENT device (cudaGetSymbolAddress; done once
 * per device, also lazily by the first hsma_direct_sum_static on that device) -- call it before starting a graph capture.
 * The first launch of a kernel on a device makes the CUDA runtime load it (lazy module loading, which may allocate inside the
 * driver): make one warm-up call of hsma_direct_sum_static with the same refine before a capture.
 */
hsma_status hsma_direct_sum_static(const double* tgt, long long T, const double* src, const double* q,
                                   long long N, const double* shift_host, const double* sign_host,
                                   const double* w_host, int C, int central_cell, long long self_offset,
                                   int refine, double* phi_out, void* cuda_stream);
hsma_status hsma_static_scratch_setup(void);
long long hsma_static_scratch_bytes(void);
/* test hook: fill the whole scratch array with `byte` on `cuda_stream` (0xFF makes every double a NaN): a call that follows must
 * still give the right answer, i.e. it reads nothing that it has not written itself. */
hsma_status hsma_static_scratch_fill(int byte, void* cuda_stream);
/* Raw kernel (c): phi[t] = sum_j Q_j/rho - P_j.(t - R_j)/rho^3.  All dev pointers; R [M,3], P [M,3]. */
hsma_status hsma_node_sum(const double* tgt, long long T, const double* R, const double* Q,
                          const double* P, long long M, double* phi_out, void* cuda_stream);
/* Raw potential+gradient kernels: as the two above, and grad_out dev [T,3] = d phi / d tgt_t.
 * phi_out may be NULL. */
hsma_status hsma_direct_field(const double* tgt, long long T, const double* src, const double* q,
                              long long N, const double* shift_host, const double* sign_host,
                              const double* w_host, int C, int central_cell, long long self_offset,
                              int refine, double* phi_out, double* grad_out, void* cuda_stream);
hsma_status hsma_node_field(const double* tgt, long long T, const double* R, const double* Q,
                            const double* P, long long M, double* phi_out, double* grad_out,
                            void* cuda_stream);

/* DFMA-only microbenchmark on the current device: sustained FP64 FMA TFLOP/s over ~`seconds`
 * (the roofline denominator).  host out; synchronises. */
hsma_status hsma_fp64_peak(double seconds, double* tflops_out, double* sm_clock_mhz_out);

/*
 * Per-stage device timing (bench.py "roofline").  While enabled, every evaluate
 * records CUDA events on the plan's stream around its stages (no host synchronisation is added).
 * hsma_plan_get_timing synchronises the stream and writes the stage durations of the LAST evaluate in
 * milliseconds to host ms_out [8]:
 *   [0] H1 pre-pass (+ neutrality)   [1] H2 near_sum_kernel over the check targets, kernel only
 *   [2] H2 finish + H3 fit + H4 map  [3] H5 near_sum_kernel over the sources, kernel only (the hot loop)
 *   [4] H6 node_sum_kernel, kernel only   [5] H7 finish + energy   [6] whole evaluate
 *   [7] near_algorithm = FMM: the far field of step (b) (M2L + L2L), which runs before step (a) and is NOT in [0] or [3]
 *       ([0] then holds the leaf sort, P2M and M2M; [3] the leaf kernel); 0 otherwise
 */
hsma_status hsma_plan_set_timing(hsma_plan* plan, int enable);
hsma_status hsma_plan_get_timing(hsma_plan* plan, double* ms_out);

/*
 * Form of step (b).  When an evaluate covers all N targets (t0 = 0, t1 = N; whole-cell near set, at
 * least 32 source tiles = N > 7936, at most 128 near cells) the targets are the sources and the image sum is
 * symmetric (every image cell has a partner of equal weight), so each unordered pair can be
 * evaluated once and feed both phi_i and phi_j (and both gradients): the "symmetric" form, near_sym_kernel /
 * near_sym_field_kernel.  form = 0 (default): automatic -- the symmetric form whenever it applies; form = 1: always
 * the ordered-pair kernel (near_sum_kernel), e.g. to compare the two; form = 2: the symmetric form wherever it applies
 * (today the same as 0; kept distinct so that a future cost model in the automatic choice cannot change a caller's request).
 * Shards (t0 > 0 or t1 < N) and the sphere-culled near set always use the ordered form.  Other values:
 * HSMA_ERR_INVALID_ARG.  hsma_plan_last_pair_form: what the last evaluate used for step (b): 1 ordered, 2 symmetric
 * (0: null plan).
 */
hsma_status hsma_plan_set_pair_form(hsma_plan* plan, int form);
int hsma_plan_last_pair_form(const hsma_plan* plan);   /* also 3: step (b) ran as the FMM (near_algorithm = HSMA_NEAR_ALG_FMM) */

/* near_algorithm = FMM: what[0] = expansion order, [1] = leaf level of the last evaluate (0 before the first), [2] = leaf
 * boxes of that level, [3] = 1 if the plan's geometry lets step (a) use the multipoles too.  host out [4].
 * HSMA_ERR_INVALID_ARG for a plan created with the direct algorithm. */
hsma_status hsma_plan_fmm_info(hsma_plan* plan, long long* what_out);

/*
 * Scratch of the symmetric form.  The unordered pairs of one rank are walked in "waves" (launches);
 * each wave keeps one column-sum line (2 KB; 8 KB with forces) per (target block, source tile) visit it makes and is
 * followed by a gather that adds its row and column sums into the near potential in a fixed order.  The number of waves
 * is chosen so that the column scratch of a wave stays below `bytes` (default and bytes = 0: 64 MiB; a wave never
 * spans fewer than 2 visits), so the plan's scratch is O(N): sources 32 B, slots 4 B, near sum 8 B (32 B with forces)
 * per source, a few partial rows, plus this cap -- not the O(N^2 / 10^6) x 2 KB of a single launch.  If the scratch
 * cannot be allocated, form 0 (automatic) falls back to the ordered-pair kernel; form 2 returns HSMA_ERR_ALLOC.
 * Results are bit-reproducible for a given (N, cap); two different caps agree to rounding (<= 1e-13 relative).
 * hsma_plan_scratch_bytes: bytes of per-evaluate scratch the plan holds right now (grown to the largest N seen).
 */
hsma_status hsma_plan_set_sym_scratch_cap(hsma_plan* plan, long long bytes);
long long hsma_plan_scratch_bytes(const hsma_plan* plan);

/*
 * Lattice-factored image sums (Eq.(3)/(4): the near set is a full box of image cells).
 * For one (target, source) pair the squared distances to all images separate over the axes, |d_k|^2 = X[k_x] + Y[k_y] +
 * Z[k_z], so the direct sums of steps (a) and (b) cost one add per image for r^2 and the charges and cell weights enter
 * once per pair.  On by default wherever it applies: whole-cell near sets of shape (1,1,1) periodic, (1,1,1) reflecting,
 * (1,1,1) and (1,1,2) xy-periodic / z-reflecting; any other cell table, the sphere-culled near set and the far-data table keep
 * the cell-by-cell kernels.  on = 0 restores those everywhere (same results to rounding: the two forms differ only in
 * the rounding of r^2).  hsma_plan_image_factoring: 1 if the factored kernels are in use for this plan.
 */
hsma_status hsma_plan_set_image_factoring(hsma_plan* plan, int on);
int hsma_plan_image_factoring(const hsma_plan* plan);

/*
 * Thread safety: a plan (and the stream it was created on) must be used by one host thread at a time; different
 * plans may be driven from different host threads (the only process-wide state, the launch counter and the
 * allocation epoch that invalidates captured graphs, is atomic).  Host synchronisation: hsma_evaluate* enqueue work
 * and return, EXCEPT that the first call at a larger N than any before grows the plan's scratch (cudaFree +
 * cudaMalloc: an implicit device synchronisation).
 */

/* total number of kernels this library has launched in this process */
long long hsma_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* HSMA_H_ */
