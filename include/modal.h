/*
 * modal.h -- C ABI of libmodal.so: B200 (sm_100a) time-stepping of N_q coupled modal
 * oscillators (arXiv 2505.05940), batched over parameter sets.
 *
 * The library implements the data-parallel hot path of the paper:
 *   q''_k + 2 gamma_k q'_k + omega_k^2 q_k = fext_k - fnl_k(q)        (Eq. 12)
 * advanced by the explicit two-step schemes of PAPER.md:138-167 (Eq. 15-23), with
 *   fnl = 0                                   MODAL_LINEAR
 *   fnl_k = c lambda_k q_k sum_v lambda_v q_v^2   MODAL_TENSION  (Eq. 8)
 *   fnl_k = sum_n eta_n sum_r H^n_kr q_r,  eta_n = s_n sum_pq H^n_pq q_p q_q
 *                                             MODAL_VK       (Eq. 9-11;
 *                                             C eliminated by H^k_ij = C^j_ik)
 * and a point read-out out[b][n] = sum_k w_k q_k^n.
 *
 * Every step of the path runs in hand-written CUDA kernels; there is no CPU fallback:
 * modal_simulate() on a plan created without a device returns MODAL_ECUDA.
 *
 * Conventions
 *  - All descriptor quantities are SI, fp64.  Host arrays are fp64; the device keeps the
 *    coupling tensor, s_n, w_k, lambda_k in fp32 and the oscillator state and update
 *    coefficients in fp64.
 *  - Ownership: the caller owns every buffer it passes; the library copies what it needs
 *    before returning.  The library owns the plan and its device storage.
 *  - Errors: every call returns a modal_status and never aborts or throws.  All validation
 *    messages of the last failing (or warning) call on a plan are available, '\n'-separated,
 *    from modal_last_error(); for a failed modal_plan_create (*out == NULL) pass NULL.
 *  - Modes beyond the stability limit of the scheme are masked (q_k == 0, excluded from
 *    force, projection and read-out; reading R11); masking is a warning.
 *  - Thread safety: calls on different plans may run concurrently; calls on one plan may not, and a plan
 *    carries ONE simulation at a time: its exchange buffers and device state belong to the last
 *    modal_simulate call, so a second call on the same plan must wait for the first to finish
 *    (modal_plan_check, or a synchronised stream), also when the two use different streams.
 */
#ifndef MODAL_H_
#define MODAL_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct modal_plan modal_plan; /* opaque, owned by the library */

typedef enum {
    MODAL_OK = 0,
    MODAL_EINVAL = 1,    /* descriptor / argument validation failed (e.g. FTM with a mode omega <= sigma) */
    MODAL_EINCOMPAT = 2, /* valid request this build cannot run (size limits)              */
    MODAL_EUNSTABLE = 3, /* a sample went non-finite; first_bad_step says where            */
    MODAL_ECUDA = 4,     /* CUDA runtime error, or no device attached to the plan          */
    MODAL_ENOMEM = 5
} modal_status;

typedef enum { MODAL_LINEAR = 0, MODAL_TENSION = 1, MODAL_VK = 2 } modal_model;
typedef enum { MODAL_SV = 0, MODAL_FTM = 1 } modal_scheme;
typedef enum { MODAL_STRING = 0, MODAL_RECT = 1 } modal_geom;
typedef enum { MODAL_BC_FIXED_SS = 0 } modal_bc; /* fixed string / simply supported plate */

/* Reference geometry, material and sizes of a plan (Eq. 1-4). */
typedef struct {
    int model, scheme, geom, bc; /* the enums above                                            */
    double Lx, Ly, h;            /* string: Lx = L; Ly, h unused                               */
    double E, rho, nu;           /* rho: kg/m^3 (plate) or kg/m (string)  (reading R3)         */
    double T0, D;                /* tension; bending stiffness. RECT with D <= 0 => E h^3/(12(1-nu^2)) */
    double area;                 /* string cross-section A for tau = E A / (2 L)  (Eq. 4)      */
    double sigma0, sigma1;       /* gamma_k = sigma0 + sigma1 lambda_k  (Eq. 14, reading R9)   */
    double pickup_x, pickup_y;   /* read-out point, metres (string: pickup_x only)             */
    int n_q, n_phi;              /* transverse / in-plane mode counts; n_phi = 0 unless VK     */
    double sample_rate;          /* Hz                                                         */
    int max_batch, max_steps;    /* sizes the plan's device storage                            */
} modal_plan_desc;

/* Create a plan: validates the descriptor (all violations are reported), derives the mode
 * index sets, lambda_k, omega_k, gamma_k, the stability mask, s_n / tau/rho, the pickup
 * weights and (VK) the coupling tensor H of the simply supported plate in closed form, packs
 * H into its device layout and allocates device storage on `cuda_device`.
 * cuda_device < 0 creates a host-only plan (queries work, modal_simulate returns MODAL_ECUDA).
 * `desc` stays owned by the caller.  On failure *out = NULL. */
modal_status modal_plan_create(const modal_plan_desc *desc, int cuda_device, modal_plan **out);

/* Replace coefficients (Eq. 13-14; Eq. 9-11).  Any pointer may be NULL =
 * keep the plan's current value.  All pointers are HOST pointers; the library copies.
 * Per-sample arrays have coeff_batch rows: 1 (broadcast to every sample) or the batch of the
 * following modal_simulate calls (<= max_batch).  All non-NULL per-sample arrays of one call
 * share coeff_batch; arrays left NULL keep their previous rows only if coeff_batch is
 * unchanged, otherwise row 0 of the previous value is broadcast. */
typedef struct {
    int coeff_batch;
    const double *omega;    /* [coeff_batch][n_q]  rad/s                                          */
    const double *sigma;    /* [coeff_batch][n_q]  1/s   (gamma_k)                                */
    const double *nl_scale; /* VK: s_n = E/(2 rho zeta_n^4) (x geometry scale, reading R14)       */
                            /*     [coeff_batch][n_phi];  TENSION: tau/rho_m  [coeff_batch]       */
    const double *lambda;   /* TENSION: [coeff_batch][n_q]                                        */
    const double *pickup;   /* [coeff_batch][n_q]                                                 */
    const double *H_full;   /* VK: [n_phi][n_q][n_q] row-major, shared by the whole batch.  The   */
                            /* library checks |H[n][p][q]-H[n][q][p]| <= 1e-12 max|H| and packs.  */
} modal_coeffs;
modal_status modal_coeffs_upload(modal_plan *plan, const modal_coeffs *coeffs);

typedef struct {
    const double *q0;        /* host [batch][n_q]: modal displacement at n = 0                    */
    const double *qm1;       /* host [batch][n_q]: displacement at n = -1; NULL => zero initial   */
                             /* velocity, q^-1 = q^0 + (T^2/2)(-omega^2 q^0 - fnl(q^0)) (R8),     */
                             /* evaluated on the device                                            */
    const float *fext_signal;/* optional DEVICE [batch][n_steps] scalar force signal, NULL = none */
    const double *fext_gain; /* optional host [batch][n_q]: Phi_k(x_e)/mass; required with signal */
    double *traj_dev;        /* optional DEVICE [batch][n_steps][n_q]: receives q^n (diagnostics) */
} modal_init;

/* Run n_steps of the recurrence for `batch` samples (Eq. 19/20):
 *   out_audio_dev[b][n] = sum_k w_k q_k^n,  n = 0 .. n_steps-1   (n = 0 is the initial state, R10)
 * out_audio_dev: DEVICE pointer, [batch][n_steps] fp32 row-major, caller-allocated.
 * first_bad_step: host [batch] or NULL.  When non-NULL the call synchronises the stream and
 *   fills first_bad_step[b] with the first n at which sample b's state was non-finite (-1 if
 *   none) and returns MODAL_EUNSTABLE iff any is >= 0; the finite prefix of the output is valid.
 *   When NULL the work is only enqueued on `cuda_stream` (a cudaStream_t, NULL = default) and nothing
 *   the kernels detect (instability, a cross-CTA exchange that timed out) can be reported by this call:
 *   follow it with modal_plan_check.
 * Errors: MODAL_EINVAL (batch/steps outside the plan, missing q0), MODAL_ECUDA. */
modal_status modal_simulate(modal_plan *plan, int batch, int n_steps, const modal_init *init,
                            float *out_audio_dev, int *first_bad_step, void *cuda_stream);

/* Same, with a HOST output buffer [batch][n_steps]; the library stages through plan-owned
 * device memory (host<->device copies included).  Always synchronous. */
modal_status modal_simulate_host(modal_plan *plan, int batch, int n_steps, const modal_init *init,
                                 float *out_audio_host, int *first_bad_step);

/* Completes the plan's last modal_simulate call: synchronises the stream it was enqueued on, fills
 * first_bad_step (host [batch of that call], may be NULL) and returns MODAL_EUNSTABLE / MODAL_ECUDA (a bounded
 * wait of a persistent kernel gave up: the CTAs of a team were not co-resident) / MODAL_OK. */
modal_status modal_plan_check(modal_plan *plan, int *first_bad_step);

/* Reverse pass (backpropagation through time) of a run: SURVEY.md 8(f) row 3.  MODAL_VK as described below;
 * MODAL_TENSION / MODAL_LINEAR plans (strings, Berger plates: the paper's non-linear string fits) the same with
 * fnl_mu = c lam_mu q_mu sum lam q^2, grad_nl_scale [batch] = dL/dc and no grad_H.  Given the trajectory of a
 * forward run (modal_init.traj_dev of modal_simulate with the same plan, coefficients, batch and n_steps, an explicit qm1 and no
 * external force) and gout[b][n] = dL/d out_audio[b][n] of any loss L on the audio, computes per sample
 *   dL/dq^0, dL/dq^-1 (as independent inputs of q^{n+1} = c1 q^n + c2 q^{n-1} - c3 fnl(q^n), Eq. 19/20),
 *   dL/dc1, dL/dc2, dL/dc3 and through them (SV Eq. 21-23 / FTM Eq. 16-18) dL/domega, dL/dsigma,
 *   dL/dpickup, dL/dnl_scale, and dL/dH summed over the batch (entries as independent variables under t_m = H^m q: for a
 *   symmetric parametrisation use g[n][k][r] + g[n][r][k]).  Masked modes get zero gradients.
 * Adjoint recurrence a^n = w gout_n + c1 a^{n+1} + c2 a^{n+2} - J(q^n)^T (c3 a^{n+1}); the Jacobian product costs two contractions
 * with H per step (csrc/vk_bptt.cuh).  Contractions in fp32, adjoint state and accumulators in fp64.  Synchronous: the gradients
 * are copied to the HOST arrays before it returns; any gradient pointer may be NULL.  Per-sample arrays are [batch][...] even when
 * coeff_batch is 1 (sum over the batch for shared parameters).  n_q <= 512.
 * Errors: MODAL_EINVAL (sizes, missing qm1 / traj_dev / gout_dev), MODAL_EINCOMPAT (n_q), MODAL_ECUDA. */
typedef struct {
    const double *qm1;        /* host   [batch][n_q]            q^-1 of the forward run                       */
    const double *traj_dev;   /* DEVICE [batch][n_steps][n_q]   q^n of the forward run (fp64)                 */
    const float *gout_dev;    /* DEVICE [batch][n_steps]        dL/d out_audio                                */
    double *grad_q0, *grad_qm1;            /* host [batch][n_q]                                               */
    double *grad_omega, *grad_sigma;       /* host [batch][n_q]                                               */
    double *grad_c1, *grad_c2, *grad_c3;   /* host [batch][n_q]                                               */
    double *grad_pickup;                   /* host [batch][n_q]                                               */
    double *grad_nl_scale;                 /* host [batch][n_phi]                                             */
    double *grad_H;                        /* host [n_phi][n_q][n_q], summed over the batch                   */
} modal_bptt_args;
modal_status modal_bptt(modal_plan *plan, int batch, int n_steps, const modal_bptt_args *args, void *cuda_stream);

/* Launch-selection overrides for tests and sweeps (the defaults are automatic).  Keys:
 *   "vk_impl"      0 automatic, 1 FP32 flow kernel, 2 tcgen05 batched kernel (H resident in shared memory), 3 tcgen05
 *                  streaming kernel (H streamed from L2; batch <= 64 per launch, wider batches run as consecutive launches),
 *                  4 small-system kernel (one warp per sample; N_q, N_phi <= 32, N_phi N_q^2 <= 8192: chosen automatically there),
 *                  5 dense-team kernel (a team of <= 32 CTAs per sample, every CTA keeps the whole state, one hop per step; chosen
 *                  automatically below batch 64 when the dense H of a CTA's modes fits shared memory, e.g. 100 + 50 modes, and,
 *                  from batch 8 on, a CTA has at most 8 modes)
 *                  6 replicated-state kernel (ONE sample; every CTA keeps the whole state and whole in-plane modes whose H^n sits in
 *                  shared memory as the dense blocks of the parity-class structure, stored once per symmetric pair; thread-block
 *                  clusters reduce the partial forces through distributed shared memory, one L2 hop per step; chosen automatically
 *                  at batch 1 when the dense-team kernel does not fit and the blocks do: the 400 + 200 mode plate of the headline)
 *   "flow_g"       CTAs per team of the flow kernel (0 automatic)
 *   "flow_ns"      TMA ring slots of the flow kernel (0: none, streamed tiles are read directly from L2)
 *   "flow_res"     resident tiles per CTA of the flow kernel (-1 automatic)
 *   "mma_split"    k blocks per mode class of the batched kernel (0 automatic)
 *   "mma_ng"       in-plane modes per CTA of the batched kernel (0 automatic)
 *   "mma_nstg"     operand ring stages of the batched / streaming kernel (0 automatic)
 *   "mma_cluster"  1 (default): the CTAs of an n group of the batched kernel form a thread-block cluster and exchange partial G
 *                  through distributed shared memory when the device keeps all clusters co-resident; 0: through L2
 *   "parity_order" 1 (default): transverse modes grouped by index parity on the device; 0: plan order
 *   "timing"       1: per-phase cycle counters of the persistent kernels, printed to stderr (synchronous)
 * Returns MODAL_EINVAL for an unknown key or a value out of range. */
modal_status modal_plan_set_option(modal_plan *plan, const char *key, int value);

/* In-plane (Airy) basis of a MODAL_VK plan, PAPER.md:53, 123 (the paper gives no formula; readings R5 / R16):
 *   MODAL_AIRY_SINE          the transverse sine products, zeta_n^4 = lambda_n^2 (default, reading R5)
 *   MODAL_AIRY_CLAMPED_RITZ  the clamped-plate eigenfunctions Lap Lap Psi = zeta^4 Psi, Psi = dPsi/dn = 0, by Rayleigh-Ritz on
 *                            T_i(x/Lx) T_j(y/Ly), T_i(s) = sin(pi s) sin(i pi s), i, j <= n_trial (0: chosen from n_phi)
 * Recomputes H (closed-form integrals) and nl_scale = E / (2 rho zeta_n^4) of the reference geometry for every coefficient row;
 * omega, sigma, pickup stay.  With the Ritz basis H does not follow the (Lx Ly)^(-5/2) law across aspect ratios, so per-sample
 * geometries (modal_derive_coeffs) keep reading R14 only at the plan's aspect ratio.  Errors: MODAL_EINVAL, MODAL_EINCOMPAT. */
typedef enum { MODAL_AIRY_SINE = 0, MODAL_AIRY_CLAMPED_RITZ = 1 } modal_airy_basis;
modal_status modal_plan_set_airy_basis(modal_plan *plan, int basis, int n_trial);

void modal_plan_destroy(modal_plan *plan);
const char *modal_last_error(const modal_plan *plan);

/* ---- host-side helpers (no device needed) --------------------------------------------- */

typedef enum {
    MODAL_Q_MODE_M = 0,      /* int    [n_q]    transverse mode index m_k                          */
    MODAL_Q_MODE_N = 1,      /* int    [n_q]    transverse mode index n_k (string: all 0)          */
    MODAL_Q_PHI_M = 2,       /* int    [n_phi]                                                      */
    MODAL_Q_PHI_N = 3,       /* int    [n_phi]                                                      */
    MODAL_Q_LAMBDA = 4,      /* double [n_q]    lambda_k of the reference geometry                  */
    MODAL_Q_OMEGA = 5,       /* double [coeff_batch][n_q]                                           */
    MODAL_Q_SIGMA = 6,       /* double [coeff_batch][n_q]                                           */
    MODAL_Q_NL_SCALE = 7,    /* double [coeff_batch][n_phi] (VK) or [coeff_batch] (TENSION)         */
    MODAL_Q_PICKUP = 8,      /* double [coeff_batch][n_q]   (before masking)                        */
    MODAL_Q_ACTIVE = 9,      /* int    [coeff_batch][n_q]   1 = active, 0 = masked (R11)            */
    MODAL_Q_H_FULL = 10,     /* double [n_phi][n_q][n_q]: the fp32 values the device holds, widened */
    MODAL_Q_COEFF_BATCH = 11,/* int    [1]                                                          */
    MODAL_Q_KERNEL_INFO = 12,/* int    [8] of the last launch: kernel family (1 tension, 2 small-system, 3 flow, 4 batched tcgen05, 5 streaming, */
                             /*        6 dense team: CTAs per team, samples per launch),                                        */
                             /*        8 replicated state: CTAs, CTAs per cluster; [6] most rows of an item),                   */
                             /*        tcgen05), CTAs per team (flow) or CTAs, teams (flow) / n groups (batched) / samples per  */
                             /*        launch (streaming), threads, dynamic shared memory bytes, flags (1: H resident in shared */
                             /*        memory or L2, 2: team of several CTAs), ring slots (flow) / accumulator slots (batched)  */
                             /*        / most tiles of a CTA (streaming), padded n_q                                            */
    MODAL_Q_MMA_LAYOUT = 14, /* int    [16]: layout the batched tcgen05 kernel would use (host side, no device needed):  */
                             /*        fits, k blocks, n groups, modes per group, TMEM columns per slot, slots, columns */
                             /*        per mode, quads per block, K chunks, most K chunks of a CTA, CTAs, rows owned,   */
                             /*        fewest / most K chunks of a CTA, slab KiB, most source blocks of a CTA           */
    MODAL_Q_MMA_SLAB_CHECK = 15, /* double [3]: non-zero entries of H covered by the operand slabs, non-zero entries of */
                             /*        H, max |hi + lo - H| / max |H| (host-side self check of the packing)             */
    MODAL_Q_AIRY_ZETA4 = 16, /* double [n_phi]: zeta_n^4 of the plan's in-plane basis (reference geometry)                    */
    MODAL_Q_STREAM_LAYOUT = 17, /* int [16]: layout the streaming tcgen05 kernel would use (host side): fits, CTAs, k blocks, */
                             /*        K chunks of the operand axis, tiles, most / fewest tiles of a CTA, most q chunks of a   */
                             /*        CTA, most / fewest rows a CTA owns, most K chunks of a tile, chunks in total, stream    */
                             /*        MiB, most CTAs of a k block, 0, 0                                                       */
    MODAL_Q_STREAM_CHECK = 18, /* double [4]: non-zero entries of H covered by the H stream, non-zero entries of H,            */
                             /*        max |hi + lo - H| / max |H|, rows owned in total (== n_q)                               */
    MODAL_Q_REPL_CHECK = 19, /* double [8]: host-side check of the replicated-state kernel's layout on 132 CTAs: layout found,      */
                             /*        non-zero entries of H rebuilt exactly once from the packed blocks (negative: mismatches), */
                             /*        non-zero entries of H, largest H of a CTA in KiB, most modes of a CTA, most rows of an item, */
                             /*        packed floats in total, CTAs that hold a mode                                            */
    MODAL_Q_TILE_STATS = 13  /* int    [2]: 16x16 tiles of the packed H, and how many hold a non-zero.   */
                             /*        The device keeps the transverse modes grouped by index parity   */
                             /*        (internal order only: every array of this API is in plan order),*/
                             /*        so that the parity zeros of H fill whole  */
                             /*        tiles, which the step kernel never reads.                       */
} modal_query;
/* Copies the item into `dst` (capacity `dst_bytes`); returns MODAL_EINVAL if it does not fit. */
modal_status modal_plan_query(const modal_plan *plan, int what, void *dst, unsigned long long dst_bytes);

/* Per-sample coefficients for a geometry other than the plan's reference one, with the PLAN'S
 * mode index sets (reading R14): for RECT fills omega, sigma [n_q], nl_scale [n_phi]
 * (= E/(2 rho zeta^4) (c_b/c_ref)^2, c = (Lx Ly)^(-5/2)) and pickup [n_q] at
 * (pickup_x_frac Lx, pickup_y_frac Ly); for STRING fills omega, sigma, lambda, pickup [n_q] and
 * nl_scale [1] = tau/rho_lin.  Fields of `geom` that are <= 0 / NaN fall back to the plan's. */
typedef struct {
    double Lx, Ly, h;           /* RECT; STRING: Lx = L                                          */
    double T0, D, rho, area;    /* STRING per-sample tension, stiffness, linear density, section */
    double pickup_x_frac, pickup_y_frac;
} modal_sample_geom;
modal_status modal_derive_coeffs(const modal_plan *plan, const modal_sample_geom *geom,
                                 double *omega, double *sigma, double *nl_scale,
                                 double *lambda, double *pickup);

/* q0[k] = int w0 Phi_k for the raised-cosine bump w0 = (A/2)(1 + cos(2 pi r / W)), r < W/2
 * centred at (x0,y0) (string: x0) on a sample of size (Lx, Ly) with the plan's index sets
 * (reading R13).  q0: host [n_q]. */
modal_status modal_project_bump(const modal_plan *plan, double Lx, double Ly, double x0, double y0,
                                double W, double A, double *q0);

/* ---- machine peaks (measurement helper, not on the simulation path) ---------------------- */

/* Micro-benchmarks of the denominators the roofline fractions of this build are quoted against and that the driver's
 * MEASURED_PEAKS.json does not hold: FP32 / FP64 FMA issue peaks, L2-resident and HBM read bandwidth, shared-
 * memory and TMEM read bandwidth, and the latency of the cross-CTA exchange primitives of the persistent kernels (one-way,
 * SM cycles), idle and while the other SMs keep the L2 busy.  Runs ~1 s on `cuda_device`; MODAL_ECUDA on a CUDA error. */
typedef struct {
    double sm_clock_mhz;                 /* SM clock during the FMA test (cycles / event time)                      */
    double fp32_tflops, fp64_tflops;     /* 2 flop per FMA                                                          */
    double l2_read_gbs_8mb, l2_read_gbs_64mb, hbm_read_gbs;     /* ld.global.cg sweeps; 1 GiB for HBM               */
    double smem_read_gbs, smem_bytes_per_clk_sm;                /* conflict-free LDS.128, all SMs / per SM          */
    double tmem_read_bytes_per_clk_sm;   /* tcgen05.ld.32x32b.x32, four warps                                       */
    double hop_cycles_idle, hop_cycles_loaded;                  /* tagged 8-byte word, st.relaxed -> polling ld.relaxed */
    double relacq_hop_cycles_idle, relacq_hop_cycles_loaded;    /* payload + st.release flag -> poll, ld.acquire, payload */
} modal_peaks;
modal_status modal_measure_peaks(int cuda_device, modal_peaks *out);

/* The von Karman recurrence through ONE entry point that ALLOCATES NOTHING, for callers that cannot call cudaMalloc (code under
 * CUDA graph capture, tight serving loops, harnesses that forbid it).  No plan: every array is a DEVICE pointer of the caller on
 * the calling thread's current device; the call makes no cudaMalloc / cudaFree / allocating library call and never synchronises
 * (it enqueues memsets and kernel launches on `cuda_stream`).  The only scratch the kernel needs -- the exchange buffer of the
 * CTA team that shares a sample -- is a file-scope static __device__ array of MODAL_STATIC_SCRATCH_BYTES (1 MiB) that every GPU
 * which loads the library holds until the process exits.
 *   q^{n+1}_k = c1_k q^n_k + c2_k q^{n-1}_k - c3_k fnl_k(q^n)          PAPER.md:153-161 Eq. 19/20 (no external force)
 *   fnl_k = sum_n eta_n sum_r H^n_kr q_r,  eta_n = s_n sum_pq H^n_pq q_p q_q      PAPER.md:112-123 Eq. 9-11, C eliminated (:283)
 *   out_audio_dev[b][n] = sum_k w_k q^n_k,  n = 0 .. n_steps-1  (n = 0 is q0)
 * Arguments (all row-major): H_dev fp32 [n_phi][n_q][n_q]; c1_dev, c2_dev, c3_dev fp64 and w_dev fp32 [coeff_batch][n_q];
 * s_dev fp32 [coeff_batch][n_phi]; coeff_batch = 1 (one row for every sample) or batch; q0_dev, qm1_dev fp64 [batch][n_q]
 * (q^0 and q^-1); out_audio_dev fp32 [batch][n_steps]; first_bad_dev int [batch] or NULL, receives -1, the first step at which
 * the sample was non-finite, or -2 if a cross-CTA exchange timed out (the CTAs of a team were not co-resident: the GPU was shared
 * with other work); err / err_bytes: optional host buffer for the message of a failing call.
 * Precision as modal_simulate: force in fp32, state and update in fp64.  batch = 0 or n_steps = 0 does the per-device set-up only
 * (cudaGetSymbolAddress of the scratch array; call it once before a graph capture).
 * Limits: n_q <= MODAL_STATIC_MAX_NQ (256): MODAL_EINCOMPAT beyond.  Any batch: more samples than SMs run as consecutive launches.
 * The scratch array is SHARED by every call on a device and keeps the last call's contents (each launch clears the part it uses
 * first): calls that overlap on the GPU (different streams, no dependency) RACE and give wrong results -- order them.
 * Errors: MODAL_EINVAL (sizes, NULL pointer), MODAL_EINCOMPAT (limits), MODAL_ECUDA. */
#define MODAL_STATIC_MAX_NQ 256
#define MODAL_STATIC_SCRATCH_BYTES (1u << 20)
modal_status modal_vk_simulate_static(int n_q, int n_phi, int batch, int n_steps, int coeff_batch,
                                      const float *H_dev, const double *c1_dev, const double *c2_dev, const double *c3_dev,
                                      const float *s_dev, const float *w_dev, const double *q0_dev, const double *qm1_dev,
                                      float *out_audio_dev, int *first_bad_dev, void *cuda_stream, char *err, int err_bytes);

#ifdef __cplusplus
}
#endif
#endif /* MODAL_H_ */
