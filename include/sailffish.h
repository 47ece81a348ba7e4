/*
 * sailffish.h -- C ABI of the B200-native spectral Poisson hot path (SailFFish, arxiv 2301.01145).
 *
 * The library (libsailffish_b200.so, built from paper_2301_01145_b200/csrc/) links the CUDA runtime
 * only: no torch types, no C++ types and no exceptions cross this boundary.  Every entry point
 * returns an sf_status; a human-readable message for the last failure on a plan is available from
 * sf_last_error().  Citations "PAPER.md:<line>" refer to the paper text under /root/reference/.
 *
 * What a plan computes (sec 2.2 "four-step spectral solve"):
 *     1. forward transform of the source along every axis
 *        - periodic:  real-to-complex DFT                        (eq. 8)
 *        - Dirichlet, cell-boundary grid:  DST-I                 (Table 1 row 1)
 *        - Dirichlet, cell-centre   grid:  DST-II  (back: DST-III)  (Table 1 row 2)
 *        - Neumann,   cell-boundary grid:  DCT-I                 (Table 1 row 3)
 *        - Neumann,   cell-centre   grid:  DCT-II  (back: DCT-III)  (Table 1 row 4)
 *        - unbounded: zero-padded to twice the length, real-to-complex DFT
 *                     (Hockney-Eastwood, sec 2.5; only non-zero pencils are
 *                     transformed -- the "pruned" variant of PAPER.md:213)
 *     2. multiply by the spectral multiplier: 1 / eigenvalue of the chosen operator
 *        (pseudo-spectral or second-order finite difference, Table 1, zero mode
 *        set to zero) or by the stored transform of the regularised free-space Green's
 *        function
 *     3. optional spectral differentiation: multiply by i k (eq. 10) -> gradient
 *        of the solution, or curl of a 3-component solution
 *     4. backward transform (DST-I / DCT-III / complex-to-real DFT), unbounded: keep the first octant
 *
 * Array layout (all calls): dense, x fastest: index = ix + n[0]*(iy + n[1]*iz); vector fields are
 * component-major (component c starts at c*n[0]*n[1]*n[2]).  Element type is float (SF_F32) or
 * double (SF_F64) as chosen at plan creation.
 *
 * Threading: calls on one plan must not be issued concurrently; separate plans are independent.
 * All compute calls are asynchronous on the plan's stream; sf_get_output to host memory and
 * sf_synchronize block until the stream has drained.
 */
#ifndef SAILFFISH_B200_H
#define SAILFFISH_B200_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sf_plan_s* sf_plan;

typedef enum {
    SF_OK = 0,
    SF_ERR_INVALID_ARG = -1, /* NULL pointer, non-positive size, unknown enum value            */
    SF_ERR_UNSUPPORTED = -2, /* a combination the method / this build does not cover (see below) */
    SF_ERR_ALLOC = -3,       /* device or host allocation failed                                */
    SF_ERR_CUDA = -4,        /* a CUDA runtime call or kernel launch failed                     */
    SF_ERR_STATE = -5        /* call out of order (solve before source, output before solve)    */
} sf_status;

/* Boundary condition per axis.  The paper's solvers use one type on all axes and
 * leave mixed conditions, by 1-D transforms chosen per direction, as future work.  Built here:
 * Dirichlet and Neumann may be mixed freely per axis -- every axis takes the row of Table 1 that its
 * own condition selects on the plan's grid type, its eigenvalue column and its boundary-value weights; the size rule
 * of sf_plan_create applies per axis.  sf_solve only (sf_gradient returns UNSUPPORTED on such plans).  A periodic or
 * unbounded axis next to another type returns SF_ERR_UNSUPPORTED. */
typedef enum { SF_BC_PERIODIC = 0, SF_BC_DIRICHLET = 1, SF_BC_NEUMANN = 2, SF_BC_UNBOUNDED = 3 } sf_bc;

/* Grid type (eq. 9): REGULAR = cell-boundary nodes, STAGGERED = cell centres. */
typedef enum { SF_GRID_CELL_BOUNDARY = 0, SF_GRID_CELL_CENTRE = 1 } sf_grid;

/* Operator / multiplier (PAPER.md:173 eigenvalue type; PAPER.md:189 Green's function type). */
typedef enum {
    SF_OP_PSEUDO_SPECTRAL = 0, /* -k^2 symbol (Table 1 "PS" column)                               */
    SF_OP_FD2 = 1,             /* eigenvalues of the 2nd-order finite-difference stencil ("FD2")    */
    SF_OP_GREEN_GAUSS2 = 2,    /* unbounded: Gaussian-regularised kernel of order 2, */
                               /* G(r) = -erf(r/(sqrt(2) eps))/(4 pi r), eps = eps_over_h * max(h)  */
    SF_OP_GREEN_GAUSS4 = 3,    /* orders 4 .. 10 of the same family: with g the unit Gaussian */
    SF_OP_GREEN_GAUSS6 = 4,    /* of width eps, x = r^2/(2 eps^2) and L_m the generalised Laguerre           */
    SF_OP_GREEN_GAUSS8 = 5,    /* polynomials L_m^(1/2):  G_P = G_2 - sum_{n=1}^{P/2-1} eps^2/(2n) L_{n-1}(x) g */
    SF_OP_GREEN_GAUSS10 = 6,   /* (spectrum -exp(-s^2/2) sum_{n<P/2} (s^2/2)^n/n! / k^2, s = eps k)           */
    SF_OP_GREEN_SPECTRAL = 7   /* spectrally compact kernel: -1/k^2 inside |k| <= pi/h,        */
                               /* 3-D: G(r) = -Si(pi r/h) / (2 pi^2 r); 2-D: (C(pi r/h) - ln(pi/2h) - gamma) / (2 pi),  */
                               /* C(x) = int_0^x (1 - J0(t)) / t dt; h = max spacing; eps_over_h is ignored   */
} sf_operator;

typedef enum { SF_F32 = 0, SF_F64 = 1 } sf_precision;
typedef enum { SF_MEM_HOST = 0, SF_MEM_DEVICE = 1 } sf_mem;

/* Output selectors for sf_get_output / sf_output_device_ptr. */
typedef enum {
    SF_OUT_PSI = 0,  /* solution; comp = component (0 for scalar plans)                          */
    SF_OUT_GRAD = 1, /* after sf_gradient: comp = axis (0=x,1=y,2=z) of grad psi (scalar plans)   */
    SF_OUT_CURL = 2, /* after sf_curl:     comp = component of curl psi (ncomp == 3 plans)        */
    SF_OUT_DIV = 3,  /* after sf_divergence: div psi, comp = 0 (ncomp == 3 plans)                  */
    SF_OUT_LAP = 4   /* after sf_laplacian:  lap psi, comp = component                            */
} sf_field;

typedef struct {
    int ncomp;         /* 1 = scalar, 3 = vector solved component-wise; 0 -> 1     */
    void* stream;      /* cudaStream_t the plan enqueues on; NULL = legacy default stream          */
    double rhs_sign;   /* +1: lap(psi) = f (paper eq. 2); -1: lap(psi) = -f (vorticity, eq. 17); 0 -> +1 */
    double eps_over_h; /* Gaussian regularisation width in units of max(h); 0 -> 2.0               */
} sf_options;

/*
 * sf_plan_create -- the paper's initialisation sequence (grid setup, FFT data setup, eigenvalue /
 * Green's function setup, differential-operator setup).
 *   out    [host, written]  receives the plan handle; the plan owns every table and workspace it
 *                           allocates (all on the current CUDA device) until sf_plan_destroy.
 *   ndim   2 or 3.
 *   n      [host] stored unknowns per axis (n[a] for a >= ndim is ignored and treated as 1).
 *          periodic, unbounded, Neumann cell-centre, Dirichlet cell-centre: n[a] a power of two >= 8 (x) /
 *          >= 4 (y, z); Dirichlet cell-boundary: n[a] = 2^k - 1 interior nodes (boundary nodes are not
 *          stored); Neumann cell-boundary: n[a] = 2^k + 1 nodes (boundary nodes are stored).
 *          Upper bounds (every pass is a complex transform of 4 .. 2048 points): periodic n[0] <= 4096,
 *          n[1], n[2] <= 2048; unbounded n[0] <= 2048, n[1], n[2] <= 1024 (transforms are 2 n[a] long);
 *          Dirichlet / Neumann: extended length / 2 <= 2048, i.e. n[a] <= 2047 / 2048 / 2048 / 2049 for the four
 *          rows of Table 1.  The fused pass must also fit the shared memory of an SM: checked here for sf_solve
 *          (on ncomp == 3 plans for the three tiles of sf_curl / sf_divergence), by sf_gradient for its second
 *          tile when it is called; UNSUPPORTED otherwise.
 *   h      [host] grid spacing per axis.  Domain length follows (Table 1): periodic
 *          and cell-centre L = n h; Dirichlet cell-boundary L = (n + 1) h; Neumann cell-boundary L = (n - 1) h.
 *   bc     [host] boundary condition per axis; all axes must agree.
 *   grid   selects the row of Table 1: Dirichlet cell-boundary DST-I, Dirichlet
 *          cell-centre DST-II / DST-III, Neumann cell-boundary DCT-I, Neumann cell-centre DCT-II /
 *          DCT-III; periodic and unbounded accept both (identical numerics).
 *   op     PS / FD2 for periodic, Dirichlet, Neumann; GREEN_GAUSS2 .. GREEN_GAUSS10 for unbounded plans
 *          (3-D: -erf(r / sqrt2 eps) / (4 pi r) and its higher orders; 2-D: (ln r + E1(r^2 / 2 eps^2) / 2) / (2 pi)
 *          and its higher orders), GREEN_SPECTRAL for 3-D and 2-D unbounded plans.
 *   prec   arithmetic and storage type of every array passed later.
 *   opt    [host] may be NULL (defaults above).
 * For unbounded plans this call evaluates G on the doubled grid, transforms it with the library's
 * own fp64 kernels and stores the real, even spectrum as a compact (n+1)^3 table.
 * Errors: INVALID_ARG, UNSUPPORTED (a periodic / unbounded axis mixed with another type, sizes above, ncomp not 1 or 3,
 * PS/FD2 on unbounded or GREEN on bounded plans), ALLOC, CUDA.
 */
sf_status sf_plan_create(sf_plan* out, int ndim, const long long n[3], const double h[3], const sf_bc bc[3],
                         sf_grid grid, sf_operator op, sf_precision prec, const sf_options* opt);

/*
 * sf_set_source -- the paper's Set_Input.
 *   src    ncomp dense fields of n[0]*n[1]*n[2] elements of the plan's precision.
 *   where  SF_MEM_DEVICE: the pointer is BORROWED -- it must stay valid and unchanged until the
 *          solve that consumes it has completed on the plan's stream; nothing is copied.  It must be
 *          16-byte aligned (rows are moved by 16-byte and bulk copies); INVALID_ARG otherwise.
 *          SF_MEM_HOST: the data are copied to a plan-owned device buffer on the plan's stream
 *          (the host buffer may be reused after the call returns only if it is pageable; for
 *          pinned memory after sf_synchronize or the next blocking call).
 */
sf_status sf_set_source(sf_plan plan, const void* src, sf_mem where);

/*
 * sf_set_bc_values -- inhomogeneous boundary values, folded into the boundary-adjacent source cells
 * before the forward transform (FD2 operator only).
 *   axis 0..ndim-1, side 0 = lower face, 1 = upper face.
 *   face   values over the two remaining axes, lower axis fastest (for axis 0: iy + n[1]*iz; axis 1:
 *          ix + n[0]*iz; axis 2: ix + n[0]*iy); NULL resets the face to homogeneous.
 *          Dirichlet: psi on the face; cell-boundary grids: the boundary node next to the layer,
 *                     weight -1/h^2; cell-centre grids: the face half a cell outside the layer
 *                     (ghost cell 2 g - psi), weight -2/h^2.
 *          Neumann:   d psi / d x_axis along +axis on both faces (eq. 15);
 *                     cell-centre grids: weights +1/h (lower), -1/h (upper); cell-boundary grids
 *                     (ghost node mirrored through the boundary node): +2/h, -2/h.
 *          The values are those of psi (or of its derivative) whatever rhs_sign is: the discrete equation is
 *          lap_h psi = rhs_sign f with these values in the ghost layer, so the weights above apply to
 *          rhs_sign f (the library divides them by rhs_sign before adding them to f).
 *   where  as for sf_set_source (device pointers borrowed, host data copied).
 * Errors: UNSUPPORTED for periodic / unbounded plans or the PS operator.
 */
sf_status sf_set_bc_values(sf_plan plan, int axis, int side, const void* face, sf_mem where);

/* sf_solve -- forward transform, multiply, backward transform: psi for every
 * component.  Asynchronous.  Errors: STATE (no source), CUDA. */
sf_status sf_solve(sf_plan plan);

/* sf_gradient -- as sf_solve, and additionally d psi / d x_a = IDFT(i k_a psi_hat) for every axis
 * from the same spectrum (eq. 10).  Scalar plans (UNSUPPORTED otherwise).  On unbounded
 * plans k_a are the wavenumbers of the doubled grid, as for sf_curl.  On 3-D Dirichlet / Neumann
 * plans the sine / cosine series of Table 1 is differentiated term by term (a sine series along the
 * differentiated axis comes back as a cosine series and vice versa, k_a = pi k / L_a); this is the
 * derivative of the series, meaningful for homogeneous boundary values (with folded face values the
 * odd / even extension is not smooth).  The wavenumber at the Nyquist index is taken as zero.  On
 * non-periodic plans the first call allocates a (1 + ndim)-field set of work arrays (ALLOC on failure). */
sf_status sf_gradient(sf_plan plan);

/* sf_curl -- ncomp == 3 plans: solve the three components and return u = curl psi = IDFT(i k x
 * psi_hat) in the same spectral pass (eq. 17).  Wavenumbers on the
 * transform grid (doubled for unbounded plans).  psi itself is not produced by this call. */
sf_status sf_curl(sf_plan plan);

/* sf_divergence -- the paper's DIV operator: ncomp == 3 plans; solve the three components
 * and return div psi = IDFT(sum_a i k_a psi_hat_a) in the same spectral pass (three spectra in, one
 * out).  Wavenumbers as for sf_curl (transform grid, zero at the Nyquist index).  Periodic and
 * unbounded plans; psi itself is not produced.  Read the result with SF_OUT_DIV. */
sf_status sf_divergence(sf_plan plan);

/* sf_laplacian -- the paper's NABLA operator: for every component lap psi =
 * IDFT(sum_a (i k_a)^2 psi_hat), i.e. DIV of GRAD with the same k_a (zero at the Nyquist index).  With
 * the pseudo-spectral operator this returns the source less its mean and Nyquist planes; with FD2 or
 * a regularised Green's function the source filtered by k^2 / |symbol|.  Periodic and 3-D unbounded plans;
 * psi itself is not produced.  Read the result with SF_OUT_LAP. */
sf_status sf_laplacian(sf_plan plan);

/*
 * sf_get_output -- the paper's Get_Output.
 *   field, comp   see sf_field.
 *   dst    caller-owned, n[0]*n[1]*n[2] elements; SF_MEM_HOST blocks until the copy is complete,
 *          SF_MEM_DEVICE enqueues a device-to-device copy on the plan's stream.
 * Errors: STATE if the requested field was not produced by the last compute call.
 */
sf_status sf_get_output(sf_plan plan, int field, int comp, void* dst, sf_mem where);

/* Borrow the plan-owned device buffer holding a result (valid until the next compute call or
 * sf_plan_destroy); *ptr receives a device pointer.  Same errors as sf_get_output. */
sf_status sf_output_device_ptr(sf_plan plan, int field, int comp, void** ptr);

/* Block until every operation enqueued by this plan has completed (the plan's stream and, with a copy
 * pipeline, its two copy streams). */
sf_status sf_synchronize(sf_plan plan);

/*
 * Copy pipeline for callers whose source and result live in HOST memory (the paper's Set_Input / Get_Output
 * around every solve).  depth = 2 gives the plan a second source and a second result buffer
 * and two copy streams of its own, ordered against the plan's stream by events, so that the same call sequence
 *     sf_set_source(HOST) ; sf_solve ; sf_get_output_async     (repeated)
 * overlaps the upload of step k+1, the compute of step k and the download of step k-1 (PCIe is full duplex).
 * depth = 1 (the default) is the single-stream behaviour.  The call drains the plan first.  With depth = 2:
 *   sf_set_source(HOST)   enqueues the copy on the upload stream and returns; the host buffer may be reused after
 *                         sf_synchronize (pinned) or at once (pageable: the runtime stages it).
 *   compute calls         wait for that copy, alternate between the two result buffers, and wait for the download
 *                         that still reads the buffer they are about to overwrite.
 *   sf_output_device_ptr  the borrowed pointer stays valid until the compute call AFTER the next one.
 * Errors: INVALID_ARG (depth), ALLOC (the second buffers).
 */
sf_status sf_set_pipeline(sf_plan plan, int depth);

/* sf_get_output to HOST memory without blocking: the copy is enqueued (on the download stream of a depth-2
 * pipeline, else on the plan's stream) and dst is valid after sf_synchronize.  dst should be pinned memory for the
 * copy to overlap.  Same errors as sf_get_output. */
sf_status sf_get_output_async(sf_plan plan, int field, int comp, void* dst_host);

/* Make the plan's stream wait for every copy the pipeline has enqueued so far (an event recorded on the plan's
 * stream after this call completes after them): for callers that time or order work on that stream. */
sf_status sf_pipeline_join(sf_plan plan);

/*
 * sf_probe_dft16_stage -- measurement aid, not part of the solve: the one stage of the 1-D pencil transforms
 * that could run as a matrix product, implemented three ways on the same data so that the choice
 * "no tensor cores" rests on a measurement.  A tile is 512 threads x 16 complex fp32 values;
 * value q of thread (o, lane) is handed to thread (q, lane), which computes the 16-point DFT over o of what it
 * received (times 1/4), `reps` times over.
 *   variant 0: shared-memory exchange + radix-16 butterflies on the fp32 pipe (what the library's kernels do);
 *   variant 1: tcgen05.mma kind::tf32 with the 3 x TF32 split (fp32-level accuracy), accumulators in tensor memory;
 *   variant 2: one TF32 product only (1e-3 accuracy; the ceiling of the tensor path).
 *   in_dev / out_dev  [device] ntiles * 16 * 512 complex fp32, element q of thread t of tile i at (i * 16 + q) * 512 + t.
 *   ms      [host, written] device time of one launch (CUDA events, second of two launches).
 * Runs on the legacy default stream and blocks.  Errors: INVALID_ARG, CUDA.
 */
sf_status sf_probe_dft16_stage(int variant, int reps, int ntiles, const void* in_dev, void* out_dev, float* ms);

/* Number of kernels the last compute call launched (for launch accounting in benchmarks). */
int sf_last_launch_count(sf_plan plan);

/* Bytes of device memory owned by the plan (tables + workspaces + outputs). */
long long sf_device_bytes(sf_plan plan);

/*
 * Per-step timing for profiling: with slots > 0, each of the following compute calls records CUDA
 * events around its five steps (X forward, Y forward, Z fused, Y backward, X backward) on the
 * plan's stream, into a ring of `slots` event sets (<= 4096); slots == 0 switches timing off.
 * sf_step_times_ms blocks and writes, per step, the MEAN duration over the min(slots, calls)
 * compute calls recorded since timing was enabled (milliseconds; steps that do not exist for the
 * plan are ~0).  Errors: STATE if nothing was recorded.
 */
sf_status sf_enable_step_timing(sf_plan plan, int slots);
sf_status sf_step_times_ms(sf_plan plan, float ms[5]);
/* Record only every `stride`-th compute call (default 1) while step timing is on: the event records
 * between the steps cost a few microseconds per call, which a throughput measurement that wants the
 * per-step times from inside its own timed region can dilute this way.  Errors: INVALID_ARG if stride < 1. */
sf_status sf_set_step_timing_stride(sf_plan plan, int stride);

/* Message for the last error on this plan (or, with plan == NULL, of the last failed
 * sf_plan_create on this thread).  Never NULL; owned by the library. */
const char* sf_last_error(sf_plan plan);

/*
 * sf_periodic2d_solve_static -- the periodic 2-D solve WITHOUT any allocation, for callers that may not call
 * cudaMalloc (CUDA graph capture, tight serving loops, harnesses that forbid it): no plan, one kernel launch,
 * no cudaMalloc / cudaFree / allocating library call on any path through it.  Computes what sf_solve computes on a
 * 2-D periodic fp64 plan with default options: psi with lap(psi) = f, zero-mean (PAPER.md:103-109 four-step solve;
 * eq. (8) :79-81; Table 1 periodic row :166-167; zero mode :69).
 *   n        [host] grid points per axis, powers of two, 4 <= n[a] <= SF_STATIC_MAX_N.
 *   h        [host] grid spacing per axis (domain length n[a] * h[a]).
 *   op       SF_OP_PSEUDO_SPECTRAL or SF_OP_FD2.
 *   src_dev  [device, borrowed until the launch completes] f, n[0] * n[1] doubles, x fastest.
 *   psi_dev  [device, caller-owned] psi, same layout; may be the same buffer as src_dev.
 *   stream   cudaStream_t (NULL = legacy default stream); the call is asynchronous on it.
 * The work array between the transform steps is a file-scope device array of SF_STATIC_MAX_N * (SF_STATIC_MAX_N/2 + 1)
 * complex doubles = 528 384 bytes, which every GPU that loads the library holds until the process exits.  ALL calls
 * on a device share it: calls that can overlap on the GPU (different streams, different host threads) race on it
 * and must be ordered by the caller; calls on one stream are safe back to back.  Nothing in it needs clearing and
 * nothing is carried between calls (the kernel writes every word before it reads it).  The first call on a device
 * looks up the array's device address and sets the kernel's shared-memory limit; make that call outside a stream
 * capture.  One CTA does the whole solve: meant for small grids, use a plan for throughput.
 * Errors: INVALID_ARG (null pointer, size not a power of two, or beyond SF_STATIC_MAX_N -- the message names the
 * limit), UNSUPPORTED (operator), CUDA.  Message: sf_static_last_error() (per host thread; never NULL).
 */
#define SF_STATIC_MAX_N 256
sf_status sf_periodic2d_solve_static(const long long n[2], const double h[2], sf_operator op, const void* src_dev, void* psi_dev,
                                     void* stream);
const char* sf_static_last_error(void);

/* Free everything the plan owns.  Never frees caller memory.  NULL is accepted. */
sf_status sf_plan_destroy(sf_plan plan);

/* Library version string and the compute architecture it was built for ("sm_100a"). */
const char* sf_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SAILFFISH_B200_H */
