/*
 * mm_b200.h -- C ABI of the B200-native micromagnetic hot path of arxiv/paper_2606_01114
 * ("Magnum.np.distributed").  One GPU, one context per mesh, every step a hand-written
 * sm_100a kernel; no cuFFT, no CPU fallback.
 *
 * Citations: PAPER.md = /root/reference/PAPER.md (line numbers), SURVEY = SURVEY.md.
 *
 * Conventions shared by every call
 * --------------------------------
 *  - Field arrays m, H, dmdt: contiguous [nx][ny][nz][3], component fastest, then z
 *    (the paper's state tensor state.m[x,y,z,c]), element type float
 *    (MM_F32) or double (MM_F64) as chosen at mm_ctx_create.  m is a dimensionless unit
 *    vector per cell, H in A/m, dmdt in 1/s, lengths in metres.
 *  - Pointers named m / H / dmdt / out are DEVICE pointers unless the function name ends
 *    in _host; device pointers must be 16-byte aligned.  double[3] arguments and the
 *    context handle are HOST pointers.
 *  - Ownership: the caller owns every device buffer including the two workspaces; the
 *    library never allocates or frees device memory (PyTorch does, in the binding).
 *    The context owns only small host-side plan data.
 *  - Execution: field/step calls enqueue kernels on the context's stream and return without
 *    synchronising (CUDA-graph capturable).  Results are deterministic, bit-identical from run to
 *    run: sums are reduced in a fixed order; the only atomics are atomicMax on the bit pattern of a
 *    non-negative real (the RKF45 error and the minimiser's largest change), whose result does not
 *    depend on the order of arrival.  mm_demag_init, the *_state and the *_host calls synchronise
 *    the stream before returning.
 *  - Errors: every call returns mm_status; nothing is thrown across the ABI.  After a
 *    non-OK status mm_last_error(ctx) holds a one-line explanation.
 *  - Sizes: every n_d must be of the form 2^a 3^b 5^c 7^d (1 included), nx, ny <= 1024, nz <= 512
 *    (MM_ERR_UNSUPPORTED_SIZE otherwise).  An axis with n_d = 1 is neither padded nor
 *    transformed (reading Q10 in DESIGN.md).
 */
#ifndef MM_B200_H
#define MM_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mm_ctx mm_ctx; /* opaque, owned by the library */

typedef enum { MM_F32 = 0, MM_F64 = 1 } mm_dtype;

typedef enum {
  MM_OK = 0,
  MM_ERR_INVALID_ARG = 1,      /* NULL / misaligned pointer, non-positive size or cell, H == m */
  MM_ERR_UNSUPPORTED_SIZE = 2, /* n_d has a prime factor above 7, or is above the planned maximum */
  MM_ERR_NOT_INITIALISED = 3,  /* workspace, material or mm_demag_init missing */
  MM_ERR_WORKSPACE = 4,        /* workspace too small */
  MM_ERR_CUDA = 5,             /* CUDA runtime / launch error, text in mm_last_error */
  MM_ERR_NOT_IMPLEMENTED = 6
} mm_status;

/* Field terms of H_eff (H_eff is a sum of terms). */
enum { MM_TERM_DEMAG = 1, MM_TERM_EXCHANGE = 2, MM_TERM_ANISOTROPY = 4, MM_TERM_ZEEMAN = 8,
       MM_TERM_DMI = 16, MM_TERM_STT = 32 };

/* Mesh of nx x ny x nz cells of size dx x dy x dz metres (Mesh(n, dx)). */
mm_status mm_ctx_create(int nx, int ny, int nz, double dx, double dy, double dz, mm_dtype dtype,
                        mm_ctx **out);
mm_status mm_ctx_destroy(mm_ctx *ctx);

/* cuda_stream: a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = default. */
mm_status mm_ctx_set_stream(mm_ctx *ctx, void *cuda_stream);

/* Bytes the caller must provide.  persistent: Fourier-space demag tensor, twiddle and index
 * tables (written by mm_demag_init, read afterwards) and the RKF45 / minimiser controller records.
 * scratch: padded spectra, H_demag, stage buffers, host-call staging.  Field and step calls
 * leave nothing in scratch that a later call reads, with ONE exception: between mm_minimize_init
 * and the last mm_minimize_step of a minimisation the previous iterate and gradient (m_{n-1},
 * g_{n-1}) live there, so scratch must not be overwritten by anyone else during a minimisation.
 * Two contexts may share one scratch buffer if their calls do not overlap in time and no
 * minimisation is in flight; persistent workspaces are never shared. */
mm_status mm_ctx_workspace_bytes(const mm_ctx *ctx, size_t *persistent, size_t *scratch);
mm_status mm_ctx_set_workspace(mm_ctx *ctx, void *persistent, size_t pbytes, void *scratch,
                               size_t sbytes);

/* Material (PAPER.md:92-100 state.material): Ms [A/m], Aex [J/m], Ku [J/m^3] with unit axis
 * (normalised internally; ignored if Ku == 0), Gilbert alpha, gamma [m/(A s)] (2.211e5). */
mm_status mm_set_material(mm_ctx *ctx, double Ms, double Aex, double Ku, const double axis[3],
                          double alpha, double gamma);
/* Uniform external field in A/m (PAPER.md:140-143 ExternalField(B/mu0)). */
mm_status mm_set_zeeman(mm_ctx *ctx, const double Hext[3]);
/* Per-cell saturation magnetisation and exchange stiffness ("inhomogeneous material
 * parameters"; eq. 2 is div(A grad M); discrete form: DESIGN.md reading Q31).  Ms_cells, A_cells:
 * DEVICE arrays [nx][ny][nz] in the context's dtype (A/m, J/m), owned by the caller and read at
 * every later call until replaced; either may be NULL (the uniform value of mm_set_material).
 *   demag: M_j = Ms_j m_j;   exchange: 2/(mu0 Ms_i) sum A_ij (m_j - m_i)/d^2 with the harmonic mean
 *   A_ij = 2 A_i A_j/(A_i + A_j);   anisotropy, DMI: with Ms_i (DMI: a neighbour with Ms_j = 0 counts
 *   as outside the mesh);   Ms_i = 0 is vacuum: those terms vanish, dm/dt = 0, m is left alone.
 * With arrays set the pointwise pass runs one cell per thread (no 128-bit vector path). */
mm_status mm_set_material_cells(mm_ctx *ctx, const void *Ms_cells, const void *A_cells);
/* Dzyaloshinskii-Moriya interaction (eq. 3):
 *   H = 2D/(mu0 Ms) sum_{k=x,y,z} e_k^DMI x dm/dk,
 * D in J/m^2, e[3 k + c] = component c of the DMI vector of direction k.  The paper's two
 * choices: interfacial e_x = (0,1,0), e_y = (-1,0,0), e_z = 0; bulk e_k = unit vector k.
 * dm/dk is the central difference over the two neighbours of the exchange stencil, a
 * neighbour outside the mesh being the cell itself (reading Q28).  Needs
 * mm_set_material first (Ms).  Enabled by MM_TERM_DMI. */
mm_status mm_set_dmi(mm_ctx *ctx, double D, const double e[9]);
/* Spin-transfer torque as a local effective field (reading Q29):
 *   H = a_damp (m x p) + a_field p,  p normalised by the library, amplitudes in A/m.
 * Enabled by MM_TERM_STT. */
mm_status mm_set_stt(mm_ctx *ctx, const double p[3], double a_damp, double a_field);
/* OR of MM_TERM_*; default DEMAG | EXCHANGE. */
mm_status mm_set_terms(mm_ctx *ctx, unsigned term_mask);

/* S0: Newell tensor (ref. 23 formula, evaluated in __float128 on the device
 * for offsets i,j,k >= 0), its exact even/odd mirror expressed as separable cos/sin
 * transforms in fp64, stored real in the layout the x pass consumes with 1/(Px Py Pz)
 * folded in.  Needs both workspaces.  Idempotent.  Synchronises. */
mm_status mm_demag_init(mm_ctx *ctx);

/* Writes the Fourier-space tensor in natural order, [6][nx'][ny'][nz'] with n_d' = n_d+1
 * (or 1 when n_d = 1), components xx yy zz xy xz yz, context dtype, unscaled: the real part
 * of the forward DFT of the mirrored tensor at kx<=nx, ky<=ny, kz<=nz.  For tests. */
mm_status mm_demag_nhat_export(mm_ctx *ctx, void *out);

/* H := H_demag(m) = -Ms * crop(IFFT(Nhat . FFT(pad(m))))   (PAPER.md:45 eq. 4, :47, :53).
 * Kernels S1..S5 of DESIGN.md.  H must not alias m. */
mm_status mm_demag_field(mm_ctx *ctx, const void *m, void *H);
/* H := 2A/(mu0 Ms) * 6-point Laplacian of m, Neumann boundary (eq. 2). */
mm_status mm_exchange_field(mm_ctx *ctx, const void *m, void *H);
/* H := sum of the enabled terms. */
mm_status mm_heff(mm_ctx *ctx, const void *m, void *H);
/* H := H_DMI(m) alone (eq. 3); same argument rules as mm_exchange_field. */
mm_status mm_dmi_field(mm_ctx *ctx, const void *m, void *H);
/* dmdt := -gamma/(1+alpha^2) [m x H_eff + alpha m x (m x H_eff)]  (eq. 1);
 * H_eff is evaluated internally and not materialised. */
mm_status mm_llg_rhs(mm_ctx *ctx, const void *m, void *dmdt);
/* One classic RK4 step of size dt [s] followed by m <- m/|m|; m updated in place
 * (fixed-step stand-in for the paper's RKF45; reading Q14). */
mm_status mm_rk_step(mm_ctx *ctx, void *m_inout, double dt);
/* n_steps RK4 steps of size dt, as mm_rk_step n_steps times (bit-identical results), enqueued as replays of
 * a CUDA graph of up to 128 steps that the library captures on first use and keeps until m_inout, dt or
 * any setting of the context changes: small meshes are bound by launch latency (the paper's own diagnosis,
 * "CPU dispatch latency", CUDA graphs named as the cure), and a replayed graph removes the
 * per-kernel launch cost.  Asynchronous on the context's stream like mm_rk_step; must not itself be called
 * while that stream is being captured (use mm_rk_step inside a capture of your own). */
mm_status mm_rk_steps(mm_ctx *ctx, void *m_inout, double dt, int n_steps);

/* Adaptive Runge-Kutta-Fehlberg 4(5) stepping (the integrator the paper supports;
 * the maximum error is reduced before the next step size is computed).  The controller state
 * (t, dt, tolerance, counters) lives on the DEVICE: mm_rkf45_step enqueues one ATTEMPT -- six
 * H_eff + LLG evaluations, the 5th-order candidate, err = max over cells and components of
 * |m5 - m4|, accept iff err <= tol, next dt = dt * min(5, max(0.2, 0.9 (tol/err)^(1/5))) clamped to
 * [dt_min, dt_max], and, if accepted, m := m5/|m5| per cell and t += dt -- without any host
 * synchronisation (CUDA-graph capturable).  A rejected attempt leaves m untouched.  Readings
 * Q23-Q26 of DESIGN.md.  mm_rkf45_init (re)sets the state; mm_rkf45_state synchronises the
 * stream and reads it back (any output pointer may be NULL). */
mm_status mm_rkf45_init(mm_ctx *ctx, double t0, double dt0, double tol, double dt_min, double dt_max);
mm_status mm_rkf45_step(mm_ctx *ctx, void *m_inout);
mm_status mm_rkf45_state(mm_ctx *ctx, double *t, double *dt_next, double *err_last, double *dt_last,
                         int *accepted_last, unsigned long long *n_accepted,
                         unsigned long long *n_rejected);

/* Barzilai-Borwein energy minimiser (PAPER.md:55, 146-148 minimizer.minimize(state); the paper
 * names the algorithm, the scheme is DESIGN.md reading Q30): steepest descent on the unit sphere,
 *   g = m x (m x H_eff);  tau = tau0 first, then (s.s)/(s.y) on odd and (s.y)/(y.y) on even
 *   iterations (s = m_n - m_{n-1}, y = g_n - g_{n-1}, summed over the mesh), tau0 when s.y <= 0,
 *   clamped to [tau_min, tau_max] (m/A);  m <- [(1 - tau^2 g^2/4) m - tau g]/(1 + tau^2 g^2/4);
 *   converged iff max |m_{n+1} - m_n| <= tol.
 * The state lives on the DEVICE: mm_minimize_step enqueues ONE iteration (one H_eff evaluation,
 * deterministic fixed-order sums, controller, update) without host synchronisation; once
 * converged, further iterations leave m and the state untouched.  mm_minimize_state
 * synchronises and reads the state back (any output pointer may be NULL).  mm_minimize runs up
 * to max_iter iterations, reading the state back every check_every iterations (the coordinated
 * stop of PAPER.md:55).  The minimiser reuses the RKF45 stage buffers: do not interleave it
 * with mm_rkf45_step on the same context without re-initialising. */
mm_status mm_minimize_init(mm_ctx *ctx, double tau0, double tau_min, double tau_max, double tol);
mm_status mm_minimize_step(mm_ctx *ctx, void *m_inout);
mm_status mm_minimize_state(mm_ctx *ctx, unsigned long long *iterations, double *tau_last, double *dm_max,
                            int *converged);
mm_status mm_minimize(mm_ctx *ctx, void *m_inout, int max_iter, int check_every,
                      unsigned long long *iterations, int *converged);

/* Same operations on HOST buffers (pageable or pinned): copies m host->device into scratch
 * staging, runs the device path, copies the result device->host, synchronises.  These are
 * what bench.py's end-to-end leg times. */
mm_status mm_demag_field_host(mm_ctx *ctx, const void *m_host, void *H_host);
mm_status mm_heff_host(mm_ctx *ctx, const void *m_host, void *H_host);
mm_status mm_llg_rhs_host(mm_ctx *ctx, const void *m_host, void *dmdt_host);
mm_status mm_rk_step_host(mm_ctx *ctx, void *m_inout_host, double dt);
/* count INDEPENDENT evaluations of mm_llg_rhs on host buffers (a parameter sweep, an ensemble): result i equals
 * mm_llg_rhs_host(m_host[i], dmdt_host[i]) bit for bit.  m_host, dmdt_host: HOST arrays of count HOST pointers to
 * [nx][ny][nz][3] buffers; an input may repeat, an output that repeats keeps the last result written to it (results
 * leave in order), outputs must not alias inputs.  Pipelined: the
 * upload of state i + 1 and the download of result i - 1 run on two copy streams of the library beside the kernels
 * of state i (PCIe is full duplex), through two staging slots per direction in scratch (the second pair is the RK4
 * stage buffers: do not run it while a captured mm_rk_steps graph is replaying).  The copies overlap only for
 * PINNED host memory; pageable buffers work but serialise.  Creates two streams and six events on first use (no
 * device memory).  Synchronises all three streams before returning; count = 0 is a no-op. */
mm_status mm_llg_rhs_host_batch(mm_ctx *ctx, const void *const *m_host, void *const *dmdt_host, int count);
/* The same pipeline for H_demag and H_eff (results equal mm_demag_field_host / mm_heff_host bit for bit). */
mm_status mm_demag_field_host_batch(mm_ctx *ctx, const void *const *m_host, void *const *H_host, int count);
mm_status mm_heff_host_batch(mm_ctx *ctx, const void *const *m_host, void *const *H_host, int count);

/* ------------------------------------------------------------------------------------------
 * Diagnostics and experiments.  Not part of the method's boundary: bench.py, the
 * tests and profiling runs use them; a simulation never needs to.
 * ------------------------------------------------------------------------------------------ */

/* Number of kernel launches the library has enqueued on this context since creation
 * (bench.py reports the difference over its timed region as gpu_launches). */
mm_status mm_ctx_launch_count(const mm_ctx *ctx, unsigned long long *count);

/* Per-kernel timing for the roofline report.  While enabled, every field/step call records
 * CUDA events on the context's stream around each kernel it enqueues (a few microseconds of
 * host time per launch; at most 8192 marks are kept between two reads).
 * mm_ctx_kernel_times synchronises the stream and returns, per kernel kind, the summed
 * duration in milliseconds and the number of launches since the last reset.  Kinds, in the order
 * the demag passes run (the transform axis depends on the path, see
 * mm_ctx_kernel_name):
 *   0 S1 first forward axis (r2c)   1 S2 forward y   2 S3 last axis fused with the tensor multiply
 *   3 S4 inverse y   4 S5 first axis inverse (c2r)   5 S6/S7 fused pointwise pass   6, 7 unused */
mm_status mm_ctx_set_profiling(mm_ctx *ctx, int enable);
mm_status mm_ctx_kernel_times(mm_ctx *ctx, int reset, double ms_sum[8],
                              unsigned long long count[8]);
/* Name of the __global__ function this context launches for kernel kind `kind` (e.g.
 * "zp_fast_kernel<float,16>"), as it appears in an ncu launch list; "" for unused kinds.
 * The returned string is static. */
const char *mm_ctx_kernel_name(const mm_ctx *ctx, int kind);

/* Tile widths of the generic z-first passes; 0 keeps the default.  Must be called before
 * mm_ctx_set_workspace. */
mm_status mm_ctx_set_tiles(mm_ctx *ctx, int bz, int by, int bk);

/* Demag path selection.  path: 0 = automatic (the x-first register-stage
 * kernels where they cover the mesh, else the same kernels on an enclosing mesh when its extra
 * cells cost less than the generic passes, else the generic z-first passes), 1 = generic passes
 * always, 2 = x-first register-stage kernels required, 3 = the shared-memory-stage mixed-radix
 * x-first kernels of demag_mixed.cu (MM_ERR_UNSUPPORTED_SIZE if the required kernels do not
 * cover the mesh).  Changes the workspace sizes: call before mm_ctx_workspace_bytes /
 * mm_ctx_set_workspace.  mm_ctx_path reports what runs: 0 generic, 1 x-first register-stage
 * kernels, 2 mixed-radix shared-memory stages, 3 x-first kernels on the enclosing mesh. */
mm_status mm_ctx_set_path(mm_ctx *ctx, int path);
mm_status mm_ctx_path(const mm_ctx *ctx, int *path);

/* Slab decomposition of the demag convolution over `ranks` ranks (1 .. 8; 0 = off), the paper's own scheme
 * (PAPER.md:30 "sharded into contiguous slabs along the x-axis", :47 "all-to-all transpose", :227), emulated on
 * ONE device: rank r owns the x planes [r nx/R, (r+1) nx/R) of m and H and the rows ky in [r rpr, (r+1) rpr),
 * rpr = ceil((ny + 1) / R), of the half spectrum and of the Fourier-space tensor (the paper's y-sharded kernel).
 * The passes run y (r2c) -> x -> z . Nhat . z^-1 -> x^-1 -> y^-1 (c2r); the forward y pass of a rank stores every
 * spectrum row straight into the buffer of its owner and the inverse y pass gathers them the same way, through
 * a per-rank pointer table: on several GPUs those are peer pointers and the two all-to-all transposes are these
 * stores and loads.  Needs a mesh the x-first kernels cover with two-stage plans along
 * x and y; call before mm_ctx_workspace_bytes / mm_ctx_set_workspace.  The result equals the unsharded path's
 * to rounding (different transform order). */
mm_status mm_ctx_set_slabs(mm_ctx *ctx, int ranks);

/* mm_demag_field for callers that cannot provide (or allocate) the scratch of the convolution at call time:
 * code inside a CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  Same operation, same
 * kernels and bit-identical result as mm_demag_field (PAPER.md:45 eq. 4, :47, :53), but the two padded spectra
 * A1, A2 live in ONE file-scope `static __device__` array of the library of
 * MM_STATIC_SCRATCH_BYTES bytes instead of the context's scratch workspace.  Every GPU that loads the library
 * holds that array until the process exits.
 *  - m, H: DEVICE pointers as for mm_demag_field, still passed by the caller.  The context must be set up as
 *    usual (mm_ctx_set_workspace, mm_set_material, mm_demag_init: the Fourier-space tensor and the twiddle
 *    tables in the persistent workspace are inputs of the call); the context's scratch workspace is not touched.
 *  - Limit: the spectra of the mesh must fit (mm_static_scratch_info reports capacity and need; 64^3 in fp32
 *    needs 19.2 MB); otherwise MM_ERR_WORKSPACE with the two numbers in mm_last_error.  Contexts with per-cell
 *    Ms, an enclosing (embedded) mesh or the slab emulation need more than the spectra: MM_ERR_NOT_IMPLEMENTED.
 *  - Allocates nothing: no cudaMalloc / cudaFree / allocating library routine on this call's path.  The
 *    array's device address is looked up once per device (cudaGetSymbolAddress, which loads the module on
 *    that device); do that outside a capture by calling mm_static_scratch_info once per device at set-up,
 *    with that device current.  The call itself looks it up too if that has not happened.
 *  - Shared state: ALL contexts and all calls on a device share the one array, which keeps the contents of the
 *    last call.  Nothing in it has to start at zero (the forward passes write every element the later passes
 *    read), so nothing is cleared.  Two calls that overlap on the GPU (different streams, or a graph replay
 *    beside a direct call) RACE on it and both results are garbage; calls on one stream are ordered and safe.
 *  - Asynchronous on the context's stream, capturable, like mm_demag_field. */
#define MM_STATIC_SCRATCH_BYTES (32u << 20)
mm_status mm_demag_field_static(mm_ctx *ctx, const void *m, void *H);
/* capacity := MM_STATIC_SCRATCH_BYTES; needed := bytes mm_demag_field_static uses for this context (0 where it
 * answers MM_ERR_NOT_IMPLEMENTED; left alone if ctx is NULL).  Either output may be NULL.  Also the set-up
 * step: resolves the static array's address for the CURRENT device.  Allocates nothing. */
mm_status mm_static_scratch_info(const mm_ctx *ctx, size_t *capacity, size_t *needed);

/* Last error text of this context (or of the last failed mm_ctx_create if ctx is NULL).
 * Not thread-safe. */
const char *mm_last_error(const mm_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* MM_B200_H */
