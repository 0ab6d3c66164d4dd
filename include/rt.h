/* rt.h -- C ABI of the B200-native batched RF ray tracer.
 *
 * The library integrates, for a batch of independent rays, the geometric-optics ray equations
 *
 *      dx/dt = -(dD/dk)/(dD/dw),      dk/dt = +(dD/dx)/(dD/dw)                 (Eq. 2-3)
 *
 * with the classical 4th-order Runge-Kutta tableau at a fixed step ("expressions of 4th order
 * Runga-Kutta ... a single kernel call"; inputs x, k, t, w; outputs the dispersion residual and the updated
 * x, k, t), D(x, k, w) being a cold-plasma dispersion function (Eq. 5-10; O-mode / X-mode
 * branches L157, L191) over a plasma equilibrium B(x), n_e(x) (splines L60).  Every step of that
 * path runs in hand-written sm_100a CUDA kernels: one thread per ray, all n_steps fused in one launch, RK4 state
 * and hand-derived gradients of D in registers.  There is NO CPU fallback: every entry point that computes
 * returns RT_ERR_CUDA when no CUDA device is usable.
 *
 * Conventions
 *   - All functions return RT_OK (0) or a negative RT_ERR_* code; they never throw and never abort.
 *     rt_last_error() returns a thread-local message for the last non-zero return on the calling thread.
 *   - "DEVICE" pointers are CUDA device pointers on the current device, owned by the caller (e.g. PyTorch tensors);
 *     buffers must not alias.  Inputs need the alignment of their element type; the sample outputs of rt_trace /
 *     rt_trace_w / rt_orbit (out_traj, out_final, out_residual / out_drift) must be 16-byte aligned: they are written
 *     with 128-bit stores.  "HOST" pointers are ordinary host memory.
 *   - Ray arrays are structure-of-arrays: x0[c*n_rays + i], c = 0..2 (x, y, z), i = ray.
 *   - Element type of every ray buffer follows `precision`: double for RT_F64, float for RT_F32.
 *   - Units are the paper's: x [m], k [rad/m], w [rad/s].  The step `dt` is given in tau = c*t metres
 *     (reading A3), i.e. the time step is dt/c seconds.  Sample times are t_s = s*save_stride*dt/c.
 *   - Calls with a `cuda_stream` enqueue work on that stream (a cudaStream_t cast to void*; NULL = the legacy
 *     default stream) and return without synchronising.
 *   - Ray status (reading A12): 0 = integrated all steps; 1 = a Runge-Kutta stage point left the
 *     equilibrium's domain, the ray is frozen at its last accepted state; 2 = a step produced a non-finite state,
 *     frozen likewise.  |D| reported at a state outside the domain is NaN.
 */
#ifndef RT_B200_RT_H
#define RT_B200_RT_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RT_OK               0
#define RT_ERR_INVALID     -1   /* bad argument (null pointer, negative size, misaligned buffer, bad enum) */
#define RT_ERR_UNSUPPORTED -2   /* combination not defined (e.g. X-mode over the unmagnetised parabolic slab) */
#define RT_ERR_CUDA        -3   /* CUDA runtime error, or no usable device */
#define RT_ERR_NOMEM       -4   /* host or device allocation failed */

/* Equilibria: B(x), n_e(x).  Definitions in DESIGN.md "Equilibria". */
typedef enum {
  RT_EQ_SLAB_PARABOLIC   = 0,  /* n_e = n_ref (1 + (x^2+y^2)/L^2), no B                    (BASELINE configs 1-2) */
  RT_EQ_SLAB_LINEAR_BR   = 1,  /* n_e = n_ref (x_foot - x)/L_ramp, B = (B0 R0 / x) z^; domain x > 0   (config 3;
                                  the unclamped linear profile of PAPER.md Eq. 4) */
  RT_EQ_TOKAMAK_CIRCULAR = 2,  /* B = grad(phi) x grad(psi) + F grad(phi), F = B0 R0, dpsi/dr = B0 r/q,
                                  q = q0 + q1 rho^2, n_e = n_ref (1-rho^2)^p_exp; domain rho < rho_max (config 4) */
  RT_EQ_GRID_RZ          = 3   /* psi(R,Z) bicubic, F(psi), n_e(psi) cubic not-a-knot splines of nodal data;
                                  domain = grid rectangle and psi in [psi_min, psi_max]    (config 5) */
} rt_eq_kind;

/* Dispersion functions (dimensionless; n = c k / w, Eq. 6; S, D, P of Eq. 8-10). */
typedef enum {
  RT_DISP_OMODE     = 0,       /* D = n^2 - 1 + wpe^2/w^2            (BASELINE config 1; electrons only) */
  RT_DISP_XMODE     = 1,       /* D = S n^2 - R L                     (reading A5) */
  RT_DISP_COLD_FULL = 2        /* D = Det(eps + n n - n^2 I)          (Eq. 5) */
} rt_disp_kind;

typedef enum { RT_F64 = 0, RT_F32 = 1 } rt_precision;

/* Plain-old-data description of an equilibrium.  Caller-owned; everything (including the nodal arrays) is copied
 * by rt_create_equilibrium.  Fields not used by `kind` are ignored. */
typedef struct rt_equilibrium_desc {
  int32_t kind;                       /* rt_eq_kind */
  int32_t nR, nZ, nPsi;               /* GRID_RZ: node counts (each >= 4) */
  double n_ref, L;                    /* n_ref [m^-3]: reference density of the three analytic kinds; L [m] */
  double x_foot, L_ramp, B0, R0;      /* [m], [m], [T], [m] */
  double a, q0, q1, p_exp, rho_max;   /* minor radius [m], 0 < a < R0; q = q0 + q1 rho^2; rho_max <= 0 means 0.98 */
  double Rmin, Rmax, Zmin, Zmax;      /* GRID_RZ: uniform node coordinates R_i = Rmin + i (Rmax-Rmin)/(nR-1) */
  double psi_min, psi_max;            /* GRID_RZ: uniform psi nodes of the two 1-D profiles */
  const double* psi_RZ;               /* HOST [nR][nZ] nodal psi, row-major (Z fastest) [T m^2] */
  const double* F_psi;                /* HOST [nPsi] nodal F = R B_phi [T m] */
  const double* ne_psi;               /* HOST [nPsi] nodal n_e [m^-3] */
  double ion_mass, ion_charge;        /* one ion species, n_i = n_e/ion_charge; ion_mass [kg] = 0: electrons only */
} rt_equilibrium_desc;

typedef struct rt_equilibrium rt_equilibrium;   /* opaque; owns its device tables and a host<->device workspace */

/* Validate and copy `desc`; for GRID_RZ fit the not-a-knot splines on the host in fp64 (reading A10) and
 * upload the cell-major coefficient tables.  *out receives the handle.  Errors: INVALID, NOMEM, CUDA. */
int rt_create_equilibrium(const rt_equilibrium_desc* desc, rt_equilibrium** out);

/* Free the handle and everything it owns.  NULL is accepted.  Waits, on the handle's own device, for the work that may still
 * use the handle: rt_trace_host's streams and the rt_trace_until loops launched through it; for RT_EQ_GRID_RZ also for the
 * whole device (kernels on the callers' streams may still read its tables).  Other handles' work is not waited for. */
int rt_destroy(rt_equilibrium* eq);

/* The hot path (Eq. 2-3): trace n_rays rays for n_steps RK4 steps of size dt.
 *   x0, k0        DEVICE [3][n_rays]   launch positions [m] and wave vectors [rad/m] (on-shell)
 *   omega         rad/s, one value per call
 *   save_stride   >= 1; used only when out_traj != NULL, and then n_steps % save_stride must be 0
 *   out_traj      DEVICE [n_saved][6][n_rays], n_saved = n_steps/save_stride + 1, rows (x,y,z,kx,ky,kz); sample 0 is
 *                 the launch state, sample s the state after s*save_stride steps; or NULL
 *   out_final     DEVICE [6][n_rays] state after n_steps; or NULL
 *   out_residual  DEVICE |D|: [n_saved][n_rays] if out_traj != NULL else [n_rays] (at the final state); or NULL
 *   out_status    DEVICE int32 [n_rays]; or NULL
 * n_rays == 0 or n_steps == 0 are valid (n_steps == 0 copies the launch state).  Errors: INVALID, UNSUPPORTED, CUDA. */
int rt_trace(const rt_equilibrium* eq, int disp, int precision, const void* x0, const void* k0, double omega,
             int64_t n_rays, int64_t n_steps, double dt, int64_t save_stride, void* out_traj, void* out_final,
             void* out_residual, int32_t* out_status, void* cuda_stream);

/* rt_trace with one frequency PER RAY ("inputs for x, k, t and w" -- w is a per-ray kernel input; frequency
 * scans).  Identical to rt_trace except
 *   omega         DEVICE double [n_rays], rad/s, each positive and finite (a ray with a bad w ends with status 2);
 *                 always double, whatever `precision` is
 * k0 and the k rows of the outputs are in rad/m at each ray's own frequency: n = c k / w_i (Eq. 6). */
int rt_trace_w(const rt_equilibrium* eq, int disp, int precision, const void* x0, const void* k0, const double* omega,
               int64_t n_rays, int64_t n_steps, double dt, int64_t save_stride, void* out_traj, void* out_final,
               void* out_residual, int32_t* out_status, void* cuda_stream);

/* The same call with HOST buffers (pageable or pinned): copies x0, k0 to the device, runs the rt_trace kernel and
 * copies the requested outputs back, pipelined over ray chunks on the handle's own streams; returns after the
 * results are in host memory.  Uses (and grows) the handle's workspace: not re-entrant per handle. */
int rt_trace_host(rt_equilibrium* eq, int disp, int precision, const void* x0, const void* k0, double omega,
                  int64_t n_rays, int64_t n_steps, double dt, int64_t save_stride, void* out_traj, void* out_final,
                  void* out_residual, int32_t* out_status);

/* rt_trace_host for callers that must not allocate device memory when they call the library.  rt_trace_host stages the
 * rays and their results in device buffers it gets from cudaMalloc (and creates two streams on first use).  Some host
 * programs cannot afford that:
 *   - a code that took all of the GPU's memory into its own pool at start-up (a simulation with a fixed arena, an ML
 *     framework's caching allocator): a cudaMalloc made behind its back fails, or succeeds only until the pool grows;
 *   - a code with a latency budget (a control loop around the ray tracer, a service with other streams in flight):
 *     cudaMalloc and cudaFree stall the whole device for a time nobody bounds;
 *   - a job whose device memory is accounted for once, before the run (a fixed slice of a shared GPU).
 * This entry point therefore takes its staging space from ONE array of RT_NOALLOC_SCRATCH_BYTES (64 MiB) that is part of
 * the library image: every GPU on which the process uses the library holds those 64 MiB from the moment the library's
 * code is loaded there until the process exits, whether or not this function is ever called.  The call itself makes no
 * cudaMalloc / cudaFree, creates no stream or event, and calls no routine that allocates.
 *
 * Arguments and results are those of rt_trace_host (HOST buffers, pageable or pinned; the same kernels, so the same
 * bits), plus
 *   cuda_stream   the stream the two copies in, the kernel and the copies out are enqueued on (NULL: the default
 *                 stream); the call waits for that stream before it returns, so the results are in host memory then.
 * The whole call has to fit in the array at once -- there is no chunking here: with es = 8 (fp64) or 4 (fp32) bytes and
 * every section rounded up to 256 bytes,
 *   6 n_rays es  +  [out_traj] 6 n_saved n_rays es  +  [out_final] 6 n_rays es  +  [out_residual] n_res n_rays es
 *                +  [out_status] 4 n_rays   <=  RT_NOALLOC_SCRATCH_BYTES
 * (config 1 of BASELINE.json, 1024 rays with all 1001 samples in fp64, takes 55 MiB; final states only: 2^19 rays in
 * fp64).  A larger call is refused with RT_ERR_INVALID and a message that states both byte counts; nothing is enqueued.
 *
 * First call on a device: the library looks up the array's device address there (cudaGetSymbolAddress, with that device
 * current) and keeps it; this may make the CUDA runtime load the library's code onto the device.  Make that first call
 * outside any stream capture, before the part of the program that must not stall.
 * The array is shared by every call made on that device in this process and still holds what the previous call left in it.
 * Nothing in it has to start at zero (the copies and the kernel write every byte that is read back), so nothing is
 * cleared.  Two calls whose GPU work overlaps -- two host threads, or two streams -- would write over each other's rays:
 * calls on one device must not run at the same time.  Other entry points never touch the array.
 * Errors: as rt_trace_host; RT_ERR_INVALID when the call does not fit; RT_ERR_CUDA. */
#define RT_NOALLOC_SCRATCH_BYTES (64ll << 20)
int rt_trace_host_noalloc(const rt_equilibrium* eq, int disp, int precision, const void* x0, const void* k0, double omega,
                          int64_t n_rays, int64_t n_steps, double dt, int64_t save_stride, void* out_traj,
                          void* out_final, void* out_residual, int32_t* out_status, void* cuda_stream);

/* Launch conditions ("fix w, x, k_y, k_z; Newton-solve ... to |D| < 1e-15; the initial guess selects
 * the root").  For each ray: given the position x0 and a unit direction dir, find |n| on D = 0 -- closed form
 * (O: n^2 = 1-X; X: n^2 = RL/S; full: root of Stix's biquadratic A n^4 - B n^2 + C, branch 0 = the root nearer P,
 * 1 = the other; reading A11) polished by at most 8 Newton steps until |D| < 1e-15 -- and write
 * k0 = |n| dir w/c.  fp64 only.
 *   x0, dir       DEVICE double [3][n]
 *   k0            DEVICE double [3][n]   (NaN where the branch is evanescent or x0 is outside the domain)
 *   D_out         DEVICE double [n] D at the returned state (signed); or NULL */
int rt_launch(const rt_equilibrium* eq, int disp, int branch, const double* x0, const double* dir, double omega,
              int64_t n, double* k0, double* D_out, void* cuda_stream);

/* rt_launch with one frequency per ray: omega DEVICE double [n]. */
int rt_launch_w(const rt_equilibrium* eq, int disp, int branch, const double* x0, const double* dir, const double* omega,
                int64_t n, double* k0, double* D_out, void* cuda_stream);

/* Launch conditions exactly as the paper states them: "choosing fixed values for w, x, k_y and k_z.  The
 * remaining value k_x is determined using a Newton method to a tolerance of |D(k, w)| < 1e-15.  Since the dispersion
 * functions are multi-valued, an initial guess for k_x selects among the possible roots."  Per ray: evaluate D and
 * dD/dk_x at the current k_x; stop if |D| < tol; otherwise k_x <- k_x - D / (dD/dk_x); at most max_iter updates.  fp64.
 *   x0            DEVICE double [3][n]
 *   k_guess       DEVICE double [3][n]: rows 1, 2 = the fixed k_y, k_z [rad/m]; row 0 = the initial guess for k_x
 *   omega         rad/s, used when omega_rays == NULL;  omega_rays  DEVICE double [n] per-ray frequencies, or NULL
 *   max_iter      0..1000 Newton updates at most;  tol > 0 (the paper's value: 1e-15)
 *   k0            DEVICE double [3][n]: (k_x at the last iterate, k_y, k_z); k_x = NaN at points outside the domain or after
 *                 a non-finite iterate.  May alias k_guess.
 *   D_out         DEVICE double [n] D at the returned state (signed; NaN with k_x); or NULL
 *   iters_out     DEVICE int32 [n]: number of updates made if |D| < tol was reached, -1 if it was not; or NULL
 * Errors: RT_ERR_INVALID (NULL / host / misaligned pointers, bad omega, n < 0, max_iter or tol out of range),
 * RT_ERR_UNSUPPORTED (dispersion not defined on the equilibrium), RT_ERR_CUDA.  Asynchronous on cuda_stream. */
int rt_launch_kx(const rt_equilibrium* eq, int disp, const double* x0, const double* k_guess, double omega,
                 const double* omega_rays, int64_t n, int max_iter, double tol, double* k0, double* D_out,
                 int32_t* iters_out, void* cuda_stream);

/* Critical-surface diagnostics at n points, e.g. the samples of a trajectory (cut-offs and resonances
 * "denote important changes in wave behavior, and the behavior of rays in their vicinity is an indication of the
 * correctness of the solution"; Fig. 3-4).  fp64.
 *   x, k          DEVICE double [3][n]
 *   omega         rad/s, used when omega_rays == NULL
 *   omega_rays    DEVICE double [n] per-point frequencies, or NULL
 *   out           DEVICE double [RT_NDIAG][n], rows:
 *                   0 n_e [m^-3]   1 |B| [T]   2 X = wpe^2/w^2   3 Y = |Wce|/w   4 S   5 D   6 P   (Eq. 8-10: eps11 = S,
 *                   eps12 = -i D, eps33 = P)   7 R = S + D   8 L = S - D   9 n_par^2 = (n.B)^2/|B|^2 (0 where B = 0)
 *                 Cut-offs: P = 0 (O-mode; X = 1 for electrons only), R = 0, L = 0.  Resonances: S = 0 (upper hybrid),
 *                 Y = 1 (cyclotron).  All rows are NaN at points outside the equilibrium's domain. */
#define RT_NDIAG 10
int rt_diagnostics(const rt_equilibrium* eq, const double* x, const double* k, double omega, const double* omega_rays,
                   int64_t n, double* out, void* cuda_stream);

/* The second ensemble workload of the same shape ("full orbit affects on particle losses", L213 "waves or
 * particles in a fusion plasmas ... a large ensemble of independent problems"): full orbits of charged particles in the
 * equilibrium's magnetic field,
 *      dx/dt = v ,    dv/dt = (q/m) v x B(x)          (Newton-Lorentz; the equilibria define no electric field)
 * integrated like the rays: classical RK4 at fixed step, all steps fused in one launch, one thread per particle, same
 * status rule (a stage point outside the domain freezes the particle: 1; non-finite state: 2) and output layouts.
 *   x0, v0        DEVICE [3][n]   positions [m], velocities [m/s]; element type per `precision`
 *   charge_over_mass   q/m [C/kg], signed (relativistic particles: pass q/(gamma m); |v| is constant in a pure B field)
 *   dt            time step [s]
 *   out_traj      DEVICE [n_steps/save_stride + 1][6][n], rows (x, y, z, vx, vy, vz); or NULL
 *   out_final     DEVICE [6][n]; or NULL
 *   out_drift     DEVICE relative kinetic-energy drift |v|^2/|v0|^2 - 1 (exactly 0 for the differential equation,
 *                 O(dt^4) for RK4 -- the orbits' analogue of the rays' |D|): [n_saved][n] if out_traj else [n]; or NULL
 *   out_status    DEVICE int32 [n]; or NULL
 * RT_ERR_UNSUPPORTED on the parabolic slab (no field). */
int rt_orbit(const rt_equilibrium* eq, int precision, const void* x0, const void* v0, double charge_over_mass, int64_t n,
             int64_t n_steps, double dt, int64_t save_stride, void* out_traj, void* out_final, void* out_drift,
             int32_t* out_status, void* cuda_stream);

/* Diagnostic evaluation of the integrand at n points (the quantities one RK4 stage computes):
 *   x, k          DEVICE [3][n]
 *   D_out         DEVICE [n]     signed D(x,k,w); NaN outside the domain; or NULL
 *   rhs_out       DEVICE [6][n]  (dx/dtau, dn/dtau), tau = c t, n = c k/w: the right-hand side the kernel integrates
 *                 (zero outside the domain); or NULL
 *   inside_out    DEVICE int32 [n]; or NULL */
int rt_rhs(const rt_equilibrium* eq, int disp, int precision, const void* x, const void* k, double omega, int64_t n,
           void* D_out, void* rhs_out, int32_t* inside_out, void* cuda_stream);

/* Device-side reductions over a residual / status pair as written by rt_trace (per-context reduction
 * kernels; L80 converge items).  residual: DEVICE [n] of `precision` (NaN entries are skipped), status: DEVICE
 * int32 [n] or NULL.  out: DEVICE double [6] = {max |D|, sum |D|, count finite, #status0, #status1, #status2}. */
int rt_reduce(int precision, const void* residual, const int32_t* status, int64_t n, double* out, void* cuda_stream);

/* The convergence workflow (section 2.3: "workflows ... can be implemented by chaining calls to evaluation
 * and reduction kernels until a tolerance is met"; L76: reduction kernels; SURVEY 8(f)-2 "stop-when-all-frozen").  The
 * ensemble is advanced in chunks of `chunk_steps` RK4 steps; after each chunk a device-side reduction counts the rays
 * still active (status 0) and takes max |D| over the rays whose |D| is finite; the loop stops after the first chunk at
 * which no ray is active, or max |D| > tol, or `max_chunks` chunks have run.  The loop is a CUDA-graph WHILE node whose
 * body is {trace kernel on the state in out_final, reduce kernel, decision kernel}: the condition is set ON THE DEVICE,
 * there is no host round trip between chunks, and the call returns as soon as the graph is enqueued on `cuda_stream`
 * (which must not be capturing).  A frozen ray stays frozen (and bit for bit unchanged) across chunks.
 *   x0, k0         DEVICE [3][n_rays] launch state (not modified)
 *   chunk_steps    >= 1;  max_chunks >= 0;  tol > 0, +inf switches the |D| criterion off
 *                  max_chunks == 0 reports the launch state: 0 chunks, the active count and max |D| of the launch state,
 *                  and reason 0 -- the stop tests are made at the end of a chunk, so none is made (not even when max |D|
 *                  at launch already exceeds tol).  n_rays == 0 with max_chunks > 0 reports 1 chunk, 0 active rays,
 *                  reason 1 (the loop's first chunk over an empty ensemble finds no active ray); with max_chunks == 0:
 *                  0 chunks, reason 0.  Both as the oracle's loop does (oracle/rt_oracle.cpp: oracle_trace_until).
 *   out_final      DEVICE [6][n_rays]: the state, advanced in place chunk by chunk; required
 *   out_residual   DEVICE [n_rays] |D| at the current state; required      out_status  DEVICE int32 [n_rays]; required
 *   out_info       DEVICE int64 [RT_UNTIL_INFO_WORDS], 8-byte aligned; on completion
 *                    [0] chunks run   [1] rays still active   [2] max |D| at the stop (bit pattern of a double)
 *                    [3] reason: 0 = max_chunks reached, 1 = every ray frozen, 2 = max |D| > tol (1 wins over 2)
 *                    [4..9] the last reduction as rt_reduce writes it (doubles);  [10..15] reserved
 * State rows hold k in rad/m; an active ray's k is re-rounded once per chunk by the exchange k <-> n = c k / w.
 * fp32: the chunks run the one-ray-per-thread kernel (as rt_trace_w does), rt_trace / rt_trace_host the packed
 * two-rays-per-thread kernel.  The two evaluate the same formulas but are not bit-identical (the compiler contracts some
 * multiply-add pairs of the scalar code): one fp32 chunk equals rt_trace over the same steps to ~2e-6 relative, not bit for
 * bit.  fp64 has one kernel: one chunk equals rt_trace exactly.
 * Errors: RT_ERR_INVALID (as rt_trace, and chunk_steps < 1, max_chunks < 0, tol not > 0, a NULL output), UNSUPPORTED, CUDA. */
#define RT_UNTIL_INFO_WORDS 16
int rt_trace_until(const rt_equilibrium* eq, int disp, int precision, const void* x0, const void* k0, double omega,
                   int64_t n_rays, int64_t chunk_steps, int64_t max_chunks, double dt, double tol, void* out_final,
                   void* out_residual, int32_t* out_status, int64_t* out_info, void* cuda_stream);

/* The measurement entry points (the roofline denominator rt_fma_peak and its instruction-shape variants) are declared in
 * include/rt_bench.h: they are part of the library, not of the ray-tracing interface. */

/* Number of kernel launches this library has enqueued on the calling process so far (for bench.py's gpu_launches).  The three
 * kernels in the body of rt_trace_until's device-side loop are counted once per call -- when they are recorded -- not once
 * per chunk: how often the loop ran is only known on the device (out_info[0]). */
int64_t rt_launch_count(void);

const char* rt_last_error(void);
const char* rt_version(void);

#ifdef __cplusplus
}
#endif
#endif /* RT_B200_RT_H */
