// rt_api.cu -- the C ABI of include/rt.h: argument checks, per-call constant folding (step a0), kernel dispatch,
// the host-buffer pipeline of rt_trace_host, and the equilibrium handle.  No arithmetic of the method runs on the host
// except the once-per-equilibrium spline fit (spline_fit.cpp) and the once-per-call folding of w into O(1) constants.
#include <cuda_runtime.h>

#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/rt.h"
#include "../../include/rt_bench.h"
#include "rt_kernels.cuh"
#include "rt_params.h"
#include "spline_fit.h"

namespace {

thread_local std::string g_err;
std::atomic<long long> g_launches{0};

int fail(int code, const std::string& msg) {
  g_err = msg;
  return code;
}
int cuda_fail(cudaError_t e, const char* what) {
  return fail(e == cudaErrorMemoryAllocation ? RT_ERR_NOMEM : RT_ERR_CUDA,
              std::string(what) + ": " + cudaGetErrorString(e));
}
#define RT_CUDA(call)                                  \
  do {                                                 \
    cudaError_t e_ = (call);                           \
    if (e_ != cudaSuccess) return cuda_fail(e_, #call); \
  } while (0)

}  // namespace

// ---- the handle ---------------------------------------------------------------------------------------------------
struct rt_equilibrium {
  rt_equilibrium_desc d;          // scalars only (nodal pointers nulled)
  double rho_max;
  double ne_scale;                // grid: nodal n_e table is stored divided by this
  // device tables (grid kind): fp64 and fp32 copies
  double* psi_pp64 = nullptr;
  double* prof_pp64 = nullptr;
  float* psi_pp32 = nullptr;
  float* prof_pp32 = nullptr;
  int device = 0;
  // rt_trace_host workspace: two pipeline slots
  cudaStream_t streams[2] = {nullptr, nullptr};
  void* slot[2] = {nullptr, nullptr};
  size_t slot_bytes = 0;
};

namespace {

template <class T>
rt::Params<T> make_params(const rt_equilibrium* eq, double omega) {
  if (sizeof(T) == 8)
    return rt::fold_params<T>(eq->d, eq->rho_max, eq->ne_scale, omega, reinterpret_cast<const T*>(eq->psi_pp64),
                              reinterpret_cast<const T*>(eq->prof_pp64));
  return rt::fold_params<T>(eq->d, eq->rho_max, eq->ne_scale, omega, reinterpret_cast<const T*>(eq->psi_pp32),
                            reinterpret_cast<const T*>(eq->prof_pp32));
}

// The grid kind's tables (and the host pipeline's workspace) live on the device that was current when they were created:
// a call made with another device current would dereference foreign memory.
// Only calls that touch that memory are checked: the analytic kinds' kernels take every constant by value, so an analytic
// handle works on any device -- except in rt_trace_host (uses_workspace), once its workspace exists.
int check_device(const rt_equilibrium* eq, bool uses_workspace = false) {
  if (!eq || !(eq->psi_pp64 || (uses_workspace && eq->slot[0]))) return RT_OK;
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail(e, "cudaGetDevice"); }
  if (dev != eq->device)
    return fail(RT_ERR_INVALID, "this equilibrium handle was created on CUDA device " + std::to_string(eq->device) +
                                    " but device " + std::to_string(dev) + " is current");
  return RT_OK;
}

int check_combo(const rt_equilibrium* eq, int disp) {
  if (!eq) return fail(RT_ERR_INVALID, "equilibrium handle is NULL");
  if (disp < RT_DISP_OMODE || disp > RT_DISP_COLD_FULL) return fail(RT_ERR_INVALID, "unknown dispersion kind");
  if (eq->d.kind == RT_EQ_SLAB_PARABOLIC && disp != RT_DISP_OMODE)
    return fail(RT_ERR_UNSUPPORTED, "the parabolic slab has no magnetic field: only RT_DISP_OMODE is defined on it");
  return check_device(eq);
}

int check_omega(double omega) {
  if (!(omega > 0.0) || !std::isfinite(omega)) return fail(RT_ERR_INVALID, "omega must be positive and finite");
  return RT_OK;
}

// kernel-side equilibrium kind: the tokamak has a specialised instantiation for p_exp = 3/2
int kernel_kind(const rt_equilibrium* eq) {
  if (eq->d.kind == RT_EQ_TOKAMAK_CIRCULAR && eq->d.p_exp != 1.5) return rt::EQ_TOKAMAK_POW;
  return eq->d.kind;
}

unsigned grid_for(long long n, int block) { return (unsigned)((n + block - 1) / block); }

// ---- dispatch over (EQ, DISP) ---------------------------------------------------------------------------------
#define RT_FOR_COMBOS(M)                                   \
  M(rt::EQ_PARABOLIC, rt::DISP_O)                          \
  M(rt::EQ_LINEAR, rt::DISP_O) M(rt::EQ_LINEAR, rt::DISP_X) M(rt::EQ_LINEAR, rt::DISP_FULL)     \
  M(rt::EQ_TOKAMAK, rt::DISP_O) M(rt::EQ_TOKAMAK, rt::DISP_X) M(rt::EQ_TOKAMAK, rt::DISP_FULL)  \
  M(rt::EQ_TOKAMAK_POW, rt::DISP_O) M(rt::EQ_TOKAMAK_POW, rt::DISP_X) M(rt::EQ_TOKAMAK_POW, rt::DISP_FULL)  \
  M(rt::EQ_GRID, rt::DISP_O) M(rt::EQ_GRID, rt::DISP_X) M(rt::EQ_GRID, rt::DISP_FULL)

// fp32, one frequency, no resume: the packed two-rays-per-thread kernels (rt_kernels.cuh) -- every analytic equilibrium, and
// the grid equilibrium with the full determinant (spline look-ups per ray in scalar arithmetic, the rest packed)
#define RT_FOR_PACKED_COMBOS(M)                            \
  M(rt::EQ_PARABOLIC, rt::DISP_O)                          \
  M(rt::EQ_LINEAR, rt::DISP_O) M(rt::EQ_LINEAR, rt::DISP_X) M(rt::EQ_LINEAR, rt::DISP_FULL)     \
  M(rt::EQ_TOKAMAK, rt::DISP_O) M(rt::EQ_TOKAMAK, rt::DISP_X) M(rt::EQ_TOKAMAK, rt::DISP_FULL)  \
  M(rt::EQ_TOKAMAK_POW, rt::DISP_O) M(rt::EQ_TOKAMAK_POW, rt::DISP_X) M(rt::EQ_TOKAMAK_POW, rt::DISP_FULL)  \
  M(rt::EQ_GRID, rt::DISP_FULL)
constexpr bool has_packed_kernel(int eq_kind, int disp) { return eq_kind != rt::EQ_GRID || disp == rt::DISP_FULL; }
int launch_trace_x2(const rt_equilibrium* eq, int disp, const rt::Params<float>& P, const rt::TraceArgs<float>& A, cudaStream_t st) {
#define M(E, D)                                                                                        \
  if (kernel_kind(eq) == (E) && disp == (D)) {                                                         \
    constexpr int block = rt::TraceShape2<E>::BLOCK;                                                   \
    rt::trace_kernel_x2<E, D><<<grid_for((A.n_rays + 1) / 2, block), block, 0, st>>>(P, A);            \
    ++g_launches;                                                                                      \
    RT_CUDA(cudaGetLastError());                                                                       \
    return RT_OK;                                                                                      \
  }
  RT_FOR_PACKED_COMBOS(M)
#undef M
  return fail(RT_ERR_UNSUPPORTED, "no packed kernel for this equilibrium / dispersion combination");
}
int launch_trace_x2(const rt_equilibrium*, int, const rt::Params<double>&, const rt::TraceArgs<double>&, cudaStream_t) {
  return fail(RT_ERR_UNSUPPORTED, "packed kernels are fp32 only");
}

template <class T>
int launch_trace(const rt_equilibrium* eq, int disp, const rt::Params<T>& P, const rt::TraceArgs<T>& A, cudaStream_t st) {
  if (A.n_rays == 0) return RT_OK;
  if (sizeof(T) == 4 && !A.omega && !A.status_in && has_packed_kernel(kernel_kind(eq), disp)) return launch_trace_x2(eq, disp, P, A, st);
#define M(E, D)                                                                            \
  if (kernel_kind(eq) == (E) && disp == (D)) {                                             \
    constexpr int block = rt::TraceShape<T, E>::BLOCK;                                     \
    if (A.omega)                                                                           \
      rt::trace_kernel<T, E, D, true><<<grid_for(A.n_rays, block), block, 0, st>>>(P, A);  \
    else if (A.status_in)                                                                  \
      rt::trace_kernel<T, E, D, false, true><<<grid_for(A.n_rays, block), block, 0, st>>>(P, A); \
    else if constexpr (!(sizeof(T) == 4 && has_packed_kernel((E), (D))))   /* fp32: the packed kernels, above */ \
      rt::trace_kernel<T, E, D, false><<<grid_for(A.n_rays, block), block, 0, st>>>(P, A); \
    ++g_launches;                                                                          \
    RT_CUDA(cudaGetLastError());                                                           \
    return RT_OK;                                                                          \
  }
  RT_FOR_COMBOS(M)
#undef M
  return fail(RT_ERR_UNSUPPORTED, "no kernel for this equilibrium / dispersion combination");
}

template <class T>
int launch_rhs(const rt_equilibrium* eq, int disp, const rt::Params<T>& P, const T* x, const T* k, long long n, T* D_out,
               T* rhs_out, int32_t* inside_out, cudaStream_t st) {
  if (n == 0) return RT_OK;
  const unsigned grid = grid_for(n, rt::AUX_BLOCK);
#define M(E, D)                                                                                        \
  if (kernel_kind(eq) == (E) && disp == (D)) {                                                              \
    rt::rhs_kernel<T, E, D><<<grid, rt::AUX_BLOCK, 0, st>>>(P, x, k, n, D_out, rhs_out, inside_out);  \
    ++g_launches;                                                                                      \
    RT_CUDA(cudaGetLastError());                                                                       \
    return RT_OK;                                                                                      \
  }
  RT_FOR_COMBOS(M)
#undef M
  return fail(RT_ERR_UNSUPPORTED, "no kernel for this equilibrium / dispersion combination");
}

int launch_launch(const rt_equilibrium* eq, int disp, const rt::Params<double>& P, int branch, const double* x0,
                  const double* dir, const double* omega, double omega_ref, long long n, double* k0, double* D_out,
                  cudaStream_t st) {
  if (n == 0) return RT_OK;
  const unsigned grid = grid_for(n, rt::AUX_BLOCK);
#define M(E, D)                                                                                                        \
  if (kernel_kind(eq) == (E) && disp == (D)) {                                                                         \
    if (omega)                                                                                                         \
      rt::launch_kernel<E, D, true><<<grid, rt::AUX_BLOCK, 0, st>>>(P, branch, x0, dir, omega, omega_ref, n, k0, D_out);  \
    else                                                                                                               \
      rt::launch_kernel<E, D, false><<<grid, rt::AUX_BLOCK, 0, st>>>(P, branch, x0, dir, omega, omega_ref, n, k0, D_out); \
    ++g_launches;                                                                                                      \
    RT_CUDA(cudaGetLastError());                                                                                       \
    return RT_OK;                                                                                                      \
  }
  RT_FOR_COMBOS(M)
#undef M
  return fail(RT_ERR_UNSUPPORTED, "no kernel for this equilibrium / dispersion combination");
}

int launch_launch_kx(const rt_equilibrium* eq, int disp, const rt::Params<double>& P, const double* x0, const double* kg,
                     const double* omega, double omega_ref, long long n, int max_iter, double tol, double* k0, double* D_out,
                     int32_t* iters_out, cudaStream_t st) {
  if (n == 0) return RT_OK;
  const unsigned grid = grid_for(n, rt::AUX_BLOCK);
#define M(E, D)                                                                                                             \
  if (kernel_kind(eq) == (E) && disp == (D)) {                                                                              \
    if (omega)                                                                                                              \
      rt::launch_kx_kernel<E, D, true><<<grid, rt::AUX_BLOCK, 0, st>>>(P, x0, kg, omega, omega_ref, n, max_iter, tol, k0,   \
                                                                       D_out, iters_out);                                   \
    else                                                                                                                    \
      rt::launch_kx_kernel<E, D, false><<<grid, rt::AUX_BLOCK, 0, st>>>(P, x0, kg, omega, omega_ref, n, max_iter, tol, k0,  \
                                                                        D_out, iters_out);                                  \
    ++g_launches;                                                                                                           \
    RT_CUDA(cudaGetLastError());                                                                                            \
    return RT_OK;                                                                                                           \
  }
  RT_FOR_COMBOS(M)
#undef M
  return fail(RT_ERR_UNSUPPORTED, "no kernel for this equilibrium / dispersion combination");
}

// Per-ray frequencies: the per-call constants are folded at this reference and rescaled per thread (rt_kernels.cuh:
// params_at_frequency).  1 rad/s keeps every folded constant finite in fp32 and needs no knowledge of the device array.
constexpr double kOmegaRefPerRay = 1.0;

// omega_rays: DEVICE [n_rays] per-ray frequencies (then `omega` is ignored), or NULL for the one frequency `omega`
template <class T>
int trace_device(const rt_equilibrium* eq, int disp, const void* x0, const void* k0, double omega,
                 const double* omega_rays, long long n_rays, long long n_steps, double dt, long long save_stride,
                 void* out_traj, void* out_final, void* out_residual, int32_t* out_status, cudaStream_t st,
                 const int32_t* status_in = nullptr) {
  const rt::Params<T> P = make_params<T>(eq, omega_rays ? kOmegaRefPerRay : omega);
  rt::TraceArgs<T> A;
  A.status_in = status_in;
  A.omega = omega_rays;
  A.omega_ref = kOmegaRefPerRay;
  A.x0 = static_cast<const T*>(x0);
  A.k0 = static_cast<const T*>(k0);
  A.traj = static_cast<T*>(out_traj);
  A.fin = static_cast<T*>(out_final);
  A.res = static_cast<T*>(out_residual);
  A.status = out_status;
  A.n_rays = n_rays;
  A.n_steps = n_steps;
  A.stride = save_stride;
  A.h = (T)dt;
  A.hh = T(0.5) * A.h; A.h3 = A.h * T(1.0 / 3.0); A.h6 = A.h * T(1.0 / 6.0);    // the same roundings the kernel used to make
  return launch_trace<T>(eq, disp, P, A, st);
}

int check_trace_args(const rt_equilibrium* eq, int disp, int precision, const void* x0, const void* k0, double omega,
                     long long n_rays, long long n_steps, double dt, long long save_stride, const void* out_traj) {
  int rc = check_combo(eq, disp);
  if (rc) return rc;
  if (precision != RT_F64 && precision != RT_F32) return fail(RT_ERR_INVALID, "unknown precision");
  if ((rc = check_omega(omega))) return rc;
  if (n_rays < 0 || n_steps < 0) return fail(RT_ERR_INVALID, "n_rays and n_steps must be >= 0");
  if (!std::isfinite(dt)) return fail(RT_ERR_INVALID, "dt must be finite");
  if (save_stride < 1) return fail(RT_ERR_INVALID, "save_stride must be >= 1");
  if (out_traj && (n_steps % save_stride) != 0)
    return fail(RT_ERR_INVALID, "n_steps must be a multiple of save_stride when out_traj is given");
  if (n_rays > 0 && (!x0 || !k0)) return fail(RT_ERR_INVALID, "x0 / k0 is NULL");
  return RT_OK;
}

// align: input arrays and the scalar outputs of the diagnostic kernels are read / written element by element and need the
// alignment of their element type; the sample outputs of rt_trace / rt_orbit are written with 128-bit stores (16).
int require_device_ptr(const void* p, const char* name, bool may_be_null, size_t align = 8) {
  if (!p) return may_be_null ? RT_OK : fail(RT_ERR_INVALID, std::string(name) + " is NULL");
  if (reinterpret_cast<uintptr_t>(p) & (align - 1))
    return fail(RT_ERR_INVALID, std::string(name) + " is not " + std::to_string(align) + "-byte aligned");
  cudaPointerAttributes at;
  cudaError_t e = cudaPointerGetAttributes(&at, p);
  if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail(e, "cudaPointerGetAttributes"); }
  if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)
    return fail(RT_ERR_INVALID, std::string(name) + " is not a device pointer (host buffers go through rt_trace_host)");
  return RT_OK;
}

template <class T>
int upload(const std::vector<double>& src, T** dst) {
  std::vector<T> tmp(src.begin(), src.end());
  RT_CUDA(cudaMalloc(reinterpret_cast<void**>(dst), tmp.size() * sizeof(T)));
  RT_CUDA(cudaMemcpy(*dst, tmp.data(), tmp.size() * sizeof(T), cudaMemcpyHostToDevice));
  return RT_OK;
}

void free_handle(rt_equilibrium* eq) {
  if (!eq) return;
  int cur = -1;
  const bool owns = eq->psi_pp64 || eq->slot[0] || eq->streams[0];
  if (owns && cudaGetDevice(&cur) == cudaSuccess && cur != eq->device) cudaSetDevice(eq->device); else cur = -1;
  cudaFree(eq->psi_pp64); cudaFree(eq->prof_pp64); cudaFree(eq->psi_pp32); cudaFree(eq->prof_pp32);
  for (int s = 0; s < 2; ++s) {
    if (eq->slot[s]) cudaFree(eq->slot[s]);
    if (eq->streams[s]) cudaStreamDestroy(eq->streams[s]);
  }
  if (cur >= 0) cudaSetDevice(cur);
  delete eq;
}

}  // namespace

namespace {
template <class T>
int orbit_device(const rt_equilibrium* eq, const void* x0, const void* v0, double qm, long long n, long long n_steps, double dt,
                 long long save_stride, void* out_traj, void* out_final, void* out_drift, int32_t* out_status, cudaStream_t st) {
  const rt::Params<T> P = make_params<T>(eq, 1.0);          // B(x) does not depend on a wave frequency
  rt::OrbitArgs<T> A;
  A.x0 = static_cast<const T*>(x0);
  A.v0 = static_cast<const T*>(v0);
  A.traj = static_cast<T*>(out_traj);
  A.fin = static_cast<T*>(out_final);
  A.drift = static_cast<T*>(out_drift);
  A.status = out_status;
  A.n = n;
  A.n_steps = n_steps;
  A.stride = save_stride;
  A.h = (T)dt;
  A.qm = (T)qm;
#define M(E)                                                                       \
  if (kernel_kind(eq) == (E) || ((E) == rt::EQ_TOKAMAK && kernel_kind(eq) == rt::EQ_TOKAMAK_POW)) {  \
    constexpr int block = rt::TraceShape<T, E>::BLOCK;                             \
    rt::orbit_kernel<T, E><<<grid_for(n, block), block, 0, st>>>(P, A);            \
    ++g_launches;                                                                  \
    RT_CUDA(cudaGetLastError());                                                   \
    return RT_OK;                                                                  \
  }
  M(rt::EQ_LINEAR) M(rt::EQ_TOKAMAK) M(rt::EQ_GRID)
#undef M
  return fail(RT_ERR_UNSUPPORTED, "no orbit kernel for this equilibrium kind");
}
}  // namespace

namespace {
// zero out[6], then one grid-stride pass over residual / status (8 blocks of 256 threads per SM at most)
int launch_reduce(int precision, const void* residual, const int32_t* status, long long n, double* out, cudaStream_t st) {
  RT_CUDA(cudaMemsetAsync(out, 0, 6 * sizeof(double), st));
  if (n == 0) return RT_OK;
  // the SM count of the device this launch goes to, asked for every time: an attribute query costs well under a microsecond,
  // is allowed during stream capture, and a cached value would be the first caller's device on a multi-GPU process
  int dev = 0, sms = 0;
  RT_CUDA(cudaGetDevice(&dev));
  RT_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  if (sms < 1) sms = 1;
  long long blocks = (n + 255) / 256;
  if (blocks > (long long)sms * 8) blocks = (long long)sms * 8;
  if (precision == RT_F64)
    rt::reduce_kernel<double><<<(unsigned)blocks, 256, 0, st>>>(static_cast<const double*>(residual), status, n, out);
  else
    rt::reduce_kernel<float><<<(unsigned)blocks, 256, 0, st>>>(static_cast<const float*>(residual), status, n, out);
  ++g_launches;
  RT_CUDA(cudaGetLastError());
  return RT_OK;
}
}  // namespace

namespace {
// rt_trace_until's graphs.  Destroying an executable graph that is still running blocks the host until it has finished
// (measured: the call took as long as the device work), so a launched graph is parked here with an event recorded behind
// it and released by a later call (or rt_destroy) once that event has completed -- the call itself never waits.
struct PendingGraph {
  cudaGraphExec_t ex;
  cudaGraph_t g;
  cudaEvent_t done;
  const rt_equilibrium* owner;     // the handle whose call launched it (its kernels may read that handle's device tables)
};
std::mutex g_pending_mu;
std::vector<PendingGraph> g_pending;

// Releases every parked graph that has finished.  wait_for != NULL (rt_destroy): the graphs launched through that handle are
// waited for; the other handles' graphs are only polled, so destroying one handle never blocks on another one's loop.
void release_finished_graphs(const rt_equilibrium* wait_for) {
  std::lock_guard<std::mutex> lock(g_pending_mu);
  size_t keep = 0;
  for (size_t i = 0; i < g_pending.size(); ++i) {
    PendingGraph& p = g_pending[i];
    const cudaError_t q = (wait_for && p.owner == wait_for) ? cudaEventSynchronize(p.done) : cudaEventQuery(p.done);
    if (q == cudaErrorNotReady) { g_pending[keep++] = p; continue; }
    if (q != cudaSuccess) cudaGetLastError();
    cudaGraphExecDestroy(p.ex);
    cudaGraphDestroy(p.g);
    cudaEventDestroy(p.done);
  }
  g_pending.resize(keep);
}

// Releases what rt_trace_until has acquired on its error paths (and the capture stream on every path).
struct UntilCleanup {
  cudaGraph_t g = nullptr;
  cudaGraphExec_t ex = nullptr;
  cudaStream_t cs = nullptr;
  cudaEvent_t done = nullptr;
  bool capturing = false;
  ~UntilCleanup() {
    if (capturing) { cudaGraph_t dead = nullptr; cudaStreamEndCapture(cs, &dead); }
    if (done) cudaEventDestroy(done);
    if (ex) cudaGraphExecDestroy(ex);
    if (g) cudaGraphDestroy(g);
    if (cs) cudaStreamDestroy(cs);
  }
};
}  // namespace

// ---- rt_trace_host_noalloc's staging space ------------------------------------------------------------------------------
// Device memory that belongs to the library image instead of coming from cudaMalloc (include/rt.h says who needs that and
// why).  Each GPU that loads this module holds the array until the process exits.  In HOST code the name below is only a
// stand-in for the symbol, not a device address: handing it to a kernel or to cudaMemcpy as if it were a pointer faults
// (or, on a machine where the GPU can reach host memory, quietly uses the wrong bytes).  Host code gets the real address
// from cudaGetSymbolAddress, once per device with that device current (noalloc_scratch below), and passes THAT on.
static __device__ __align__(256) unsigned char g_noalloc_scratch[RT_NOALLOC_SCRATCH_BYTES];

namespace {
constexpr int kNoallocMaxDevices = 64;
std::mutex g_noalloc_mu;
void* g_noalloc_ptr[kNoallocMaxDevices] = {};          // the array's device address on each device; NULL = not looked up yet

// The array's address on the CURRENT device.  The first call per device does the look-up (and may thereby make the runtime
// load the module there); later calls only read the table.
int noalloc_scratch(unsigned char** out) {
  int dev = -1;
  RT_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kNoallocMaxDevices)
    return fail(RT_ERR_UNSUPPORTED, "rt_trace_host_noalloc: device ordinal " + std::to_string(dev) + " is beyond the " +
                                        std::to_string(kNoallocMaxDevices) + " devices this entry point keeps an address for");
  std::lock_guard<std::mutex> lock(g_noalloc_mu);
  if (!g_noalloc_ptr[dev]) {
    void* p = nullptr;
    RT_CUDA(cudaGetSymbolAddress(&p, g_noalloc_scratch));
    if (!p) return fail(RT_ERR_CUDA, "cudaGetSymbolAddress returned a NULL address for the staging array");
    g_noalloc_ptr[dev] = p;
  }
  *out = static_cast<unsigned char*>(g_noalloc_ptr[dev]);
  return RT_OK;
}
}  // namespace

// ==== C ABI ===========================================================================================================
extern "C" {

const char* rt_last_error(void) { return g_err.c_str(); }
const char* rt_version(void) { return "rt-b200 0.1 (sm_100a)"; }
int64_t rt_launch_count(void) { return (int64_t)g_launches.load(); }

int rt_create_equilibrium(const rt_equilibrium_desc* desc, rt_equilibrium** out) {
  if (!desc || !out) return fail(RT_ERR_INVALID, "desc / out is NULL");
  *out = nullptr;
  const rt_equilibrium_desc& d = *desc;
  auto bad = [](double v) { return !std::isfinite(v); };
  if (d.kind < RT_EQ_SLAB_PARABOLIC || d.kind > RT_EQ_GRID_RZ) return fail(RT_ERR_INVALID, "unknown equilibrium kind");
  if (bad(d.ion_mass) || d.ion_mass < 0.0) return fail(RT_ERR_INVALID, "ion_mass must be >= 0");
  if (d.ion_mass > 0.0 && !(d.ion_charge > 0.0 && std::isfinite(d.ion_charge)))
    return fail(RT_ERR_INVALID, "ion_charge must be > 0 when ion_mass > 0");
  if (d.kind != RT_EQ_GRID_RZ && (bad(d.n_ref) || d.n_ref < 0.0)) return fail(RT_ERR_INVALID, "n_ref must be >= 0");
  switch (d.kind) {
    case RT_EQ_SLAB_PARABOLIC:
      if (!(d.L > 0.0) || bad(d.L)) return fail(RT_ERR_INVALID, "parabolic slab: L must be > 0");
      break;
    case RT_EQ_SLAB_LINEAR_BR:
      if (bad(d.x_foot) || bad(d.L_ramp) || d.L_ramp == 0.0) return fail(RT_ERR_INVALID, "linear slab: bad x_foot / L_ramp");
      if (bad(d.B0) || bad(d.R0) || d.B0 * d.R0 == 0.0) return fail(RT_ERR_INVALID, "linear slab: B0 R0 must be non-zero");
      break;
    case RT_EQ_TOKAMAK_CIRCULAR:
      if (!(d.a > 0.0) || !(d.R0 > 0.0) || bad(d.a) || bad(d.R0)) return fail(RT_ERR_INVALID, "tokamak: a, R0 must be > 0");
      if (bad(d.B0) || d.B0 == 0.0) return fail(RT_ERR_INVALID, "tokamak: B0 must be non-zero");
      if (bad(d.q0) || bad(d.q1) || !(d.q0 > 0.0) || d.q1 < 0.0) return fail(RT_ERR_INVALID, "tokamak: need q0 > 0, q1 >= 0");
      if (bad(d.p_exp) || d.p_exp < 1.0) return fail(RT_ERR_INVALID, "tokamak: p_exp must be >= 1");
      if (bad(d.rho_max) || d.rho_max >= 1.0) return fail(RT_ERR_INVALID, "tokamak: rho_max must be < 1");
      if (!(d.a < d.R0)) return fail(RT_ERR_INVALID, "tokamak: need a < R0 (the domain rho < rho_max must exclude R = 0)");
      break;
    default:
      if (d.nR < 4 || d.nZ < 4 || d.nPsi < 4) return fail(RT_ERR_INVALID, "grid: nR, nZ, nPsi must each be >= 4");
      if (d.nR > 16384 || d.nZ > 16384 || d.nPsi > (1 << 24)) return fail(RT_ERR_INVALID, "grid: too many nodes");
      if (bad(d.Rmin) || bad(d.Rmax) || bad(d.Zmin) || bad(d.Zmax) || !(d.Rmax > d.Rmin) || !(d.Zmax > d.Zmin) || !(d.Rmin > 0.0))
        return fail(RT_ERR_INVALID, "grid: need 0 < Rmin < Rmax and Zmin < Zmax");
      if (bad(d.psi_min) || bad(d.psi_max) || !(d.psi_max > d.psi_min)) return fail(RT_ERR_INVALID, "grid: need psi_min < psi_max");
      if (!d.psi_RZ || !d.F_psi || !d.ne_psi) return fail(RT_ERR_INVALID, "grid: nodal arrays are NULL");
  }
  rt_equilibrium* eq = new (std::nothrow) rt_equilibrium();
  if (!eq) return fail(RT_ERR_NOMEM, "out of host memory");
  eq->d = d;
  eq->d.psi_RZ = eq->d.F_psi = eq->d.ne_psi = nullptr;
  eq->rho_max = (d.rho_max > 0.0) ? d.rho_max : 0.98;
  eq->ne_scale = 1.0;
  if (d.kind == RT_EQ_GRID_RZ) {
    try {
      const size_t nn = (size_t)d.nR * d.nZ;
      for (size_t i = 0; i < nn; ++i)
        if (bad(d.psi_RZ[i])) { delete eq; return fail(RT_ERR_INVALID, "grid: psi_RZ has a non-finite entry"); }
      double nmax = 0.0;
      for (int i = 0; i < d.nPsi; ++i) {
        if (bad(d.F_psi[i]) || bad(d.ne_psi[i])) { delete eq; return fail(RT_ERR_INVALID, "grid: profile has a non-finite entry"); }
        nmax = std::fmax(nmax, std::fabs(d.ne_psi[i]));
      }
      eq->ne_scale = nmax > 0.0 ? nmax : 1.0;
      // node coordinates: R_i = Rmin + i hR (the kernels recompute them the same way)
      const double hR = (d.Rmax - d.Rmin) / (d.nR - 1), hZ = (d.Zmax - d.Zmin) / (d.nZ - 1);
      const double hP = (d.psi_max - d.psi_min) / (d.nPsi - 1);
      std::vector<double> R(d.nR), Z(d.nZ), Pn(d.nPsi), ne_n(d.nPsi);
      for (int i = 0; i < d.nR; ++i) R[i] = d.Rmin + i * hR;
      for (int i = 0; i < d.nZ; ++i) Z[i] = d.Zmin + i * hZ;
      for (int i = 0; i < d.nPsi; ++i) { Pn[i] = d.psi_min + i * hP; ne_n[i] = d.ne_psi[i] / eq->ne_scale; }
      std::vector<double> psi_pp;
      rt::fit_bicubic_not_a_knot(R.data(), Z.data(), d.psi_RZ, d.nR, d.nZ, psi_pp);
      const int nPc = d.nPsi - 1;
      std::vector<double> fpp((size_t)nPc * 4), gpp((size_t)nPc * 4), prof((size_t)nPc * 8);
      rt::fit_cubic_not_a_knot(Pn.data(), d.F_psi, 1, d.nPsi, fpp.data());
      rt::fit_cubic_not_a_knot(Pn.data(), ne_n.data(), 1, d.nPsi, gpp.data());
      for (int i = 0; i < nPc; ++i)
        for (int m = 0; m < 4; ++m) { prof[(size_t)i * 8 + m] = fpp[(size_t)i * 4 + m]; prof[(size_t)i * 8 + 4 + m] = gpp[(size_t)i * 4 + m]; }
      cudaError_t e = cudaGetDevice(&eq->device);
      if (e != cudaSuccess) { delete eq; return cuda_fail(e, "cudaGetDevice"); }
      int rc;
      if ((rc = upload<double>(psi_pp, &eq->psi_pp64)) || (rc = upload<double>(prof, &eq->prof_pp64)) ||
          (rc = upload<float>(psi_pp, &eq->psi_pp32)) || (rc = upload<float>(prof, &eq->prof_pp32))) {
        free_handle(eq);
        return rc;
      }
    } catch (const std::bad_alloc&) {
      free_handle(eq);
      return fail(RT_ERR_NOMEM, "out of host memory while fitting the splines");
    }
  }
  *out = eq;
  return RT_OK;
}

int rt_destroy(rt_equilibrium* eq) {
  if (!eq) return RT_OK;
  // with the HANDLE's device current (not whichever the caller happens to have): wait for what may still use the handle's
  // memory -- its own two streams (rt_trace_host), the convergence loops launched through it, and, for the grid kind, the
  // kernels that callers' streams may still be running against its device tables (those streams are unknown here, hence the
  // device-wide wait for that kind only).  An analytic handle owns no device memory that a kernel reads: no device-wide wait.
  int cur = -1;
  const bool owns = eq->psi_pp64 || eq->slot[0] || eq->streams[0];
  const bool switched = owns && cudaGetDevice(&cur) == cudaSuccess && cur != eq->device && cudaSetDevice(eq->device) == cudaSuccess;
  for (int s = 0; s < 2; ++s)
    if (eq->streams[s]) cudaStreamSynchronize(eq->streams[s]);
  if (eq->psi_pp64) cudaDeviceSynchronize();
  release_finished_graphs(eq);
  free_handle(eq);
  if (switched) cudaSetDevice(cur);
  return RT_OK;
}

int rt_trace(const rt_equilibrium* eq, int disp, int precision, const void* x0, const void* k0, double omega,
             int64_t n_rays, int64_t n_steps, double dt, int64_t save_stride, void* out_traj, void* out_final,
             void* out_residual, int32_t* out_status, void* cuda_stream) {
  int rc = check_trace_args(eq, disp, precision, x0, k0, omega, n_rays, n_steps, dt, save_stride, out_traj);
  if (rc) return rc;
  if (n_rays == 0) return RT_OK;
  const size_t es = (precision == RT_F64) ? 8 : 4;
  if ((rc = require_device_ptr(x0, "x0", false, es)) || (rc = require_device_ptr(k0, "k0", false, es)) ||
      (rc = require_device_ptr(out_traj, "out_traj", true, 16)) || (rc = require_device_ptr(out_final, "out_final", true, 16)) ||
      (rc = require_device_ptr(out_residual, "out_residual", true, 16)) ||
      (rc = require_device_ptr(out_status, "out_status", true, 4)))
    return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (precision == RT_F64)
    return trace_device<double>(eq, disp, x0, k0, omega, nullptr, n_rays, n_steps, dt, save_stride, out_traj, out_final, out_residual, out_status, st);
  return trace_device<float>(eq, disp, x0, k0, omega, nullptr, n_rays, n_steps, dt, save_stride, out_traj, out_final, out_residual, out_status, st);
}

int rt_trace_w(const rt_equilibrium* eq, int disp, int precision, const void* x0, const void* k0, const double* omega,
               int64_t n_rays, int64_t n_steps, double dt, int64_t save_stride, void* out_traj, void* out_final,
               void* out_residual, int32_t* out_status, void* cuda_stream) {
  int rc = check_trace_args(eq, disp, precision, x0, k0, 1.0, n_rays, n_steps, dt, save_stride, out_traj);
  if (rc) return rc;
  if (n_rays == 0) return RT_OK;
  const size_t es = (precision == RT_F64) ? 8 : 4;
  if ((rc = require_device_ptr(x0, "x0", false, es)) || (rc = require_device_ptr(k0, "k0", false, es)) ||
      (rc = require_device_ptr(omega, "omega", false)) ||
      (rc = require_device_ptr(out_traj, "out_traj", true, 16)) || (rc = require_device_ptr(out_final, "out_final", true, 16)) ||
      (rc = require_device_ptr(out_residual, "out_residual", true, 16)) ||
      (rc = require_device_ptr(out_status, "out_status", true, 4)))
    return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (precision == RT_F64)
    return trace_device<double>(eq, disp, x0, k0, 0.0, omega, n_rays, n_steps, dt, save_stride, out_traj, out_final, out_residual, out_status, st);
  return trace_device<float>(eq, disp, x0, k0, 0.0, omega, n_rays, n_steps, dt, save_stride, out_traj, out_final, out_residual, out_status, st);
}

int rt_orbit(const rt_equilibrium* eq, int precision, const void* x0, const void* v0, double charge_over_mass, int64_t n,
             int64_t n_steps, double dt, int64_t save_stride, void* out_traj, void* out_final, void* out_drift,
             int32_t* out_status, void* cuda_stream) {
  if (!eq) return fail(RT_ERR_INVALID, "equilibrium handle is NULL");
  if (eq->d.kind == RT_EQ_SLAB_PARABOLIC)
    return fail(RT_ERR_UNSUPPORTED, "the parabolic slab has no magnetic field: orbits are not defined on it");
  if (int rcd = check_device(eq)) return rcd;
  if (precision != RT_F64 && precision != RT_F32) return fail(RT_ERR_INVALID, "unknown precision");
  if (!std::isfinite(charge_over_mass)) return fail(RT_ERR_INVALID, "charge_over_mass must be finite");
  if (n < 0 || n_steps < 0) return fail(RT_ERR_INVALID, "n and n_steps must be >= 0");
  if (!std::isfinite(dt)) return fail(RT_ERR_INVALID, "dt must be finite");
  if (save_stride < 1) return fail(RT_ERR_INVALID, "save_stride must be >= 1");
  if (out_traj && (n_steps % save_stride) != 0)
    return fail(RT_ERR_INVALID, "n_steps must be a multiple of save_stride when out_traj is given");
  if (n == 0) return RT_OK;
  int rc;
  const size_t es = (precision == RT_F64) ? 8 : 4;
  if ((rc = require_device_ptr(x0, "x0", false, es)) || (rc = require_device_ptr(v0, "v0", false, es)) ||
      (rc = require_device_ptr(out_traj, "out_traj", true, 16)) || (rc = require_device_ptr(out_final, "out_final", true, 16)) ||
      (rc = require_device_ptr(out_drift, "out_drift", true, 16)) || (rc = require_device_ptr(out_status, "out_status", true, 4)))
    return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (precision == RT_F64)
    return orbit_device<double>(eq, x0, v0, charge_over_mass, n, n_steps, dt, save_stride, out_traj, out_final, out_drift, out_status, st);
  return orbit_device<float>(eq, x0, v0, charge_over_mass, n, n_steps, dt, save_stride, out_traj, out_final, out_drift, out_status, st);
}

int rt_trace_host(rt_equilibrium* eq, int disp, int precision, const void* x0, const void* k0, double omega,
                  int64_t n_rays, int64_t n_steps, double dt, int64_t save_stride, void* out_traj, void* out_final,
                  void* out_residual, int32_t* out_status) {
  int rc = check_trace_args(eq, disp, precision, x0, k0, omega, n_rays, n_steps, dt, save_stride, out_traj);
  if (rc) return rc;
  if (n_rays == 0) return RT_OK;
  if ((rc = check_device(eq, true))) return rc;
  const size_t es = (precision == RT_F64) ? 8 : 4;
  const long long n_saved = out_traj ? n_steps / save_stride + 1 : 0;
  const long long n_res = out_residual ? (out_traj ? n_saved : 1) : 0;
  // bytes per ray in a pipeline slot
  const size_t per_ray = 6 * es + (size_t)n_saved * 6 * es + (out_final ? 6 * es : 0) + (size_t)n_res * es + (out_status ? 4 : 0);
  // chunk: ~8 chunks per call, a multiple of 1024 rays, at least 2^15 rays, at most 4 GiB per slot
  long long C = ((n_rays + 7) / 8 + 1023) / 1024 * 1024;
  if (C < 32768) C = 32768;
  const long long cap = (long long)(((size_t)4 << 30) / per_ray) / 1024 * 1024;
  if (C > cap) C = cap > 1024 ? cap : 1024;
  if (C > n_rays) C = (n_rays + 1023) / 1024 * 1024;
  const size_t need = per_ray * (size_t)C + 256;
  if (!eq->streams[0]) {
    if (!eq->psi_pp64) RT_CUDA(cudaGetDevice(&eq->device));      // analytic kinds: the workspace's device
    for (int s = 0; s < 2; ++s) RT_CUDA(cudaStreamCreateWithFlags(&eq->streams[s], cudaStreamNonBlocking));
  }
  // nothing else runs on the handle's two streams: waiting for them (not for the device) is enough before the workspace
  // is reallocated, and before returning on an error path while copies into the caller's buffers may still be in flight
  auto drain = [&]() { cudaStreamSynchronize(eq->streams[0]); cudaStreamSynchronize(eq->streams[1]); };
  if (eq->slot_bytes < need) {
    drain();
    for (int s = 0; s < 2; ++s) {
      if (eq->slot[s]) { cudaFree(eq->slot[s]); eq->slot[s] = nullptr; }
    }
    eq->slot_bytes = 0;
    for (int s = 0; s < 2; ++s) RT_CUDA(cudaMalloc(&eq->slot[s], need));
    eq->slot_bytes = need;
  }
#define RT_CUDA_DRAIN(call)                                           \
  do {                                                                \
    cudaError_t e_ = (call);                                          \
    if (e_ != cudaSuccess) { drain(); return cuda_fail(e_, #call); }  \
  } while (0)
  const char* hx = static_cast<const char*>(x0);
  const char* hk = static_cast<const char*>(k0);
  int j = 0;
  for (long long off = 0; off < n_rays; off += C, ++j) {
    const long long c = (n_rays - off < C) ? (n_rays - off) : C;
    cudaStream_t st = eq->streams[j & 1];
    char* base = static_cast<char*>(eq->slot[j & 1]);
    char* dx = base;                 base += 3 * (size_t)C * es;
    char* dk = base;                 base += 3 * (size_t)C * es;
    char* dtraj = base;              base += (size_t)n_saved * 6 * (size_t)C * es;
    char* dfin = base;               base += (out_final ? 6 : 0) * (size_t)C * es;
    char* dres = base;               base += (size_t)n_res * (size_t)C * es;
    char* dstat = base;
    const size_t w = (size_t)c * es, hp = (size_t)n_rays * es;
    RT_CUDA_DRAIN(cudaMemcpy2DAsync(dx, w, hx + (size_t)off * es, hp, w, 3, cudaMemcpyHostToDevice, st));
    RT_CUDA_DRAIN(cudaMemcpy2DAsync(dk, w, hk + (size_t)off * es, hp, w, 3, cudaMemcpyHostToDevice, st));
    void* t = out_traj ? dtraj : nullptr;
    void* f = out_final ? dfin : nullptr;
    void* r = out_residual ? dres : nullptr;
    int32_t* s = out_status ? reinterpret_cast<int32_t*>(dstat) : nullptr;
    if (precision == RT_F64)
      rc = trace_device<double>(eq, disp, dx, dk, omega, nullptr, c, n_steps, dt, save_stride, t, f, r, s, st);
    else
      rc = trace_device<float>(eq, disp, dx, dk, omega, nullptr, c, n_steps, dt, save_stride, t, f, r, s, st);
    if (rc) { drain(); return rc; }
    if (out_traj)
      RT_CUDA_DRAIN(cudaMemcpy2DAsync(static_cast<char*>(out_traj) + (size_t)off * es, hp, dtraj, w, w, (size_t)n_saved * 6, cudaMemcpyDeviceToHost, st));
    if (out_final)
      RT_CUDA_DRAIN(cudaMemcpy2DAsync(static_cast<char*>(out_final) + (size_t)off * es, hp, dfin, w, w, 6, cudaMemcpyDeviceToHost, st));
    if (out_residual)
      RT_CUDA_DRAIN(cudaMemcpy2DAsync(static_cast<char*>(out_residual) + (size_t)off * es, hp, dres, w, w, (size_t)n_res, cudaMemcpyDeviceToHost, st));
    if (out_status)
      RT_CUDA_DRAIN(cudaMemcpyAsync(out_status + off, dstat, (size_t)c * 4, cudaMemcpyDeviceToHost, st));
  }
#undef RT_CUDA_DRAIN
  RT_CUDA(cudaStreamSynchronize(eq->streams[0]));
  RT_CUDA(cudaStreamSynchronize(eq->streams[1]));
  return RT_OK;
}

// rt_trace_host without a single allocation (include/rt.h): the rays and their results are staged in g_noalloc_scratch,
// the whole call at once, on the caller's stream.  Nothing here may call cudaMalloc / cudaFree or create a stream or event.
int rt_trace_host_noalloc(const rt_equilibrium* eq, int disp, int precision, const void* x0, const void* k0, double omega,
                          int64_t n_rays, int64_t n_steps, double dt, int64_t save_stride, void* out_traj,
                          void* out_final, void* out_residual, int32_t* out_status, void* cuda_stream) {
  int rc = check_trace_args(eq, disp, precision, x0, k0, omega, n_rays, n_steps, dt, save_stride, out_traj);
  if (rc) return rc;
  if (n_rays == 0) return RT_OK;
  const size_t es = (precision == RT_F64) ? 8 : 4;
  const long long n_saved = out_traj ? n_steps / save_stride + 1 : 0;
  const long long n_res = out_residual ? (out_traj ? n_saved : 1) : 0;
  const long long cap = RT_NOALLOC_SCRATCH_BYTES;
  // sections of the array, each starting on a 256-byte boundary (the kernel writes its samples with 128-bit stores)
  auto padded = [](size_t bytes) { return (bytes + 255) / 256 * 256; };
  size_t need = 0;
  bool fits = n_rays <= cap && n_saved <= cap;              // keeps the products below inside 64 bits
  size_t off_k = 0, off_traj = 0, off_fin = 0, off_res = 0, off_stat = 0;
  if (fits) {
    const size_t row3 = padded(3 * (size_t)n_rays * es);
    off_k = row3;
    off_traj = off_k + row3;
    off_fin = off_traj + padded((size_t)n_saved * 6 * (size_t)n_rays * es);
    off_res = off_fin + (out_final ? padded(6 * (size_t)n_rays * es) : 0);
    off_stat = off_res + padded((size_t)n_res * (size_t)n_rays * es);
    need = off_stat + (out_status ? padded((size_t)n_rays * 4) : 0);
    fits = need <= (size_t)cap;
  }
  if (!fits)
    return fail(RT_ERR_INVALID,
                "rt_trace_host_noalloc: this call needs " + (need ? std::to_string(need) : std::string("far more than 2^26")) +
                    " bytes of device staging space but the library's static array holds RT_NOALLOC_SCRATCH_BYTES = " +
                    std::to_string(cap) + "; trace fewer rays or samples per call, or use rt_trace_host (which allocates)");
  unsigned char* base = nullptr;
  if ((rc = noalloc_scratch(&base))) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  void* dx = base;
  void* dk = base + off_k;
  void* t = out_traj ? base + off_traj : nullptr;
  void* f = out_final ? base + off_fin : nullptr;
  void* r = out_residual ? base + off_res : nullptr;
  int32_t* s = out_status ? reinterpret_cast<int32_t*>(base + off_stat) : nullptr;
  // from the first enqueued copy on, an error return first waits for the stream: a copy into the caller's buffers may
  // still be in flight
#define RT_CUDA_WAIT(call)                                                                \
  do {                                                                                    \
    cudaError_t e_ = (call);                                                              \
    if (e_ != cudaSuccess) { cudaStreamSynchronize(st); return cuda_fail(e_, #call); }    \
  } while (0)
  const size_t in_bytes = 3 * (size_t)n_rays * es;
  RT_CUDA_WAIT(cudaMemcpyAsync(dx, x0, in_bytes, cudaMemcpyHostToDevice, st));
  RT_CUDA_WAIT(cudaMemcpyAsync(dk, k0, in_bytes, cudaMemcpyHostToDevice, st));
  if (precision == RT_F64)
    rc = trace_device<double>(eq, disp, dx, dk, omega, nullptr, n_rays, n_steps, dt, save_stride, t, f, r, s, st);
  else
    rc = trace_device<float>(eq, disp, dx, dk, omega, nullptr, n_rays, n_steps, dt, save_stride, t, f, r, s, st);
  if (rc) { cudaStreamSynchronize(st); return rc; }
  if (out_traj)
    RT_CUDA_WAIT(cudaMemcpyAsync(out_traj, t, (size_t)n_saved * 6 * (size_t)n_rays * es, cudaMemcpyDeviceToHost, st));
  if (out_final) RT_CUDA_WAIT(cudaMemcpyAsync(out_final, f, 6 * (size_t)n_rays * es, cudaMemcpyDeviceToHost, st));
  if (out_residual)
    RT_CUDA_WAIT(cudaMemcpyAsync(out_residual, r, (size_t)n_res * (size_t)n_rays * es, cudaMemcpyDeviceToHost, st));
  if (out_status) RT_CUDA_WAIT(cudaMemcpyAsync(out_status, s, (size_t)n_rays * 4, cudaMemcpyDeviceToHost, st));
#undef RT_CUDA_WAIT
  RT_CUDA(cudaStreamSynchronize(st));
  return RT_OK;
}

int rt_trace_until(const rt_equilibrium* eq, int disp, int precision, const void* x0, const void* k0, double omega,
                   int64_t n_rays, int64_t chunk_steps, int64_t max_chunks, double dt, double tol, void* out_final,
                   void* out_residual, int32_t* out_status, int64_t* out_info, void* cuda_stream) {
  int rc = check_trace_args(eq, disp, precision, x0, k0, omega, n_rays, chunk_steps, dt, 1, nullptr);
  if (rc) return rc;
  if (chunk_steps < 1) return fail(RT_ERR_INVALID, "chunk_steps must be >= 1");
  if (max_chunks < 0) return fail(RT_ERR_INVALID, "max_chunks must be >= 0");
  if (!(tol > 0.0)) return fail(RT_ERR_INVALID, "tol must be > 0 (+inf switches the |D| criterion off)");
  const size_t es = (precision == RT_F64) ? 8 : 4;
  if ((rc = require_device_ptr(out_info, "out_info", false, 8))) return rc;
  if (n_rays > 0 &&
      ((rc = require_device_ptr(x0, "x0", false, es)) || (rc = require_device_ptr(k0, "k0", false, es)) ||
       (rc = require_device_ptr(out_final, "out_final", false, 16)) ||
       (rc = require_device_ptr(out_residual, "out_residual", false, 16)) ||
       (rc = require_device_ptr(out_status, "out_status", false, 4))))
    return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  long long* info = reinterpret_cast<long long*>(out_info);
  double* red = reinterpret_cast<double*>(info + 4);
  if (n_rays == 0) {                               // an empty ensemble: the loop's first chunk (if one may run) finds no
    RT_CUDA(cudaMemsetAsync(info, 0, RT_UNTIL_INFO_WORDS * 8, st));      // active ray -- 1 chunk, "every ray frozen"
    rt::until_decide_kernel<<<1, 1, 0, st>>>(info, tol, max_chunks, 0, max_chunks > 0 ? 1 : 0);
    ++g_launches;
    RT_CUDA(cudaGetLastError());
    return RT_OK;
  }
  char* fin = static_cast<char*>(out_final);
  const size_t row3 = 3 * (size_t)n_rays * es;
  auto chunk = [&](long long steps, cudaStream_t s, const int32_t* status_in) -> int {
    const void* xs = status_in ? fin : x0;
    const void* ks = status_in ? fin + row3 : k0;
    if (precision == RT_F64)
      return trace_device<double>(eq, disp, xs, ks, omega, nullptr, n_rays, steps, dt, 1, nullptr, out_final, out_residual,
                                  out_status, s, status_in);
    return trace_device<float>(eq, disp, xs, ks, omega, nullptr, n_rays, steps, dt, 1, nullptr, out_final, out_residual,
                               out_status, s, status_in);
  };
  if (max_chunks == 0) {                           // report the launch state: one zero-step pass, reduce, record
    RT_CUDA(cudaMemsetAsync(info, 0, RT_UNTIL_INFO_WORDS * 8, st));
    if ((rc = chunk(0, st, nullptr))) return rc;
    if ((rc = launch_reduce(precision, out_residual, out_status, n_rays, red, st))) return rc;
    rt::until_decide_kernel<<<1, 1, 0, st>>>(info, tol, 0, 0, 0);
    ++g_launches;
    RT_CUDA(cudaGetLastError());
    return RT_OK;
  }
  // graph:  {copy x0, k0 into out_final; zero out_status and out_info}  ->  WHILE (cond) { chunk; reduce; decide }
  release_finished_graphs(nullptr);
  UntilCleanup u;
  RT_CUDA(cudaGraphCreate(&u.g, 0));
  cudaGraphNode_t pro[4];
  RT_CUDA(cudaGraphAddMemcpyNode1D(&pro[0], u.g, nullptr, 0, fin, x0, row3, cudaMemcpyDeviceToDevice));
  RT_CUDA(cudaGraphAddMemcpyNode1D(&pro[1], u.g, nullptr, 0, fin + row3, k0, row3, cudaMemcpyDeviceToDevice));
  cudaMemsetParams ms = {};
  ms.dst = out_status; ms.value = 0; ms.elementSize = 4; ms.width = (size_t)n_rays; ms.height = 1;
  RT_CUDA(cudaGraphAddMemsetNode(&pro[2], u.g, nullptr, 0, &ms));
  ms.dst = info; ms.width = RT_UNTIL_INFO_WORDS * 2;
  RT_CUDA(cudaGraphAddMemsetNode(&pro[3], u.g, nullptr, 0, &ms));
  cudaGraphConditionalHandle cond;
  RT_CUDA(cudaGraphConditionalHandleCreate(&cond, u.g, 1, cudaGraphCondAssignDefault));
  cudaGraphNodeParams np = {};
  np.type = cudaGraphNodeTypeConditional;
  np.conditional.handle = cond;
  np.conditional.type = cudaGraphCondTypeWhile;
  np.conditional.size = 1;
  cudaGraphNode_t loop;
  RT_CUDA(cudaGraphAddNode(&loop, u.g, pro, 4, &np));
  cudaGraph_t body = np.conditional.phGraph_out[0];
  RT_CUDA(cudaStreamCreateWithFlags(&u.cs, cudaStreamNonBlocking));
  RT_CUDA(cudaStreamBeginCaptureToGraph(u.cs, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal));
  u.capturing = true;
  if ((rc = chunk(chunk_steps, u.cs, out_status))) return rc;
  if ((rc = launch_reduce(precision, out_residual, out_status, n_rays, red, u.cs))) return rc;
  rt::until_decide_kernel<<<1, 1, 0, u.cs>>>(info, tol, max_chunks, cond, 3);
  ++g_launches;
  RT_CUDA(cudaGetLastError());
  u.capturing = false;
  RT_CUDA(cudaStreamEndCapture(u.cs, nullptr));
  RT_CUDA(cudaGraphInstantiate(&u.ex, u.g, 0));
  RT_CUDA(cudaEventCreateWithFlags(&u.done, cudaEventDisableTiming));
  RT_CUDA(cudaGraphLaunch(u.ex, st));
  RT_CUDA(cudaEventRecord(u.done, st));
  {
    std::lock_guard<std::mutex> lock(g_pending_mu);
    g_pending.push_back({u.ex, u.g, u.done, eq});
  }
  u.ex = nullptr; u.g = nullptr; u.done = nullptr;        // now owned by the pending list
  return RT_OK;
}

int rt_launch(const rt_equilibrium* eq, int disp, int branch, const double* x0, const double* dir, double omega,
              int64_t n, double* k0, double* D_out, void* cuda_stream) {
  int rc = check_combo(eq, disp);
  if (rc) return rc;
  if ((rc = check_omega(omega))) return rc;
  if (branch != 0 && branch != 1) return fail(RT_ERR_INVALID, "branch must be 0 or 1");
  if (n < 0) return fail(RT_ERR_INVALID, "n must be >= 0");
  if (n == 0) return RT_OK;
  if ((rc = require_device_ptr(x0, "x0", false)) || (rc = require_device_ptr(dir, "dir", false)) ||
      (rc = require_device_ptr(k0, "k0", false)) || (rc = require_device_ptr(D_out, "D_out", true)))
    return rc;
  const rt::Params<double> P = make_params<double>(eq, omega);
  return launch_launch(eq, disp, P, branch, x0, dir, nullptr, omega, n, k0, D_out, static_cast<cudaStream_t>(cuda_stream));
}

int rt_launch_w(const rt_equilibrium* eq, int disp, int branch, const double* x0, const double* dir, const double* omega,
                int64_t n, double* k0, double* D_out, void* cuda_stream) {
  int rc = check_combo(eq, disp);
  if (rc) return rc;
  if (branch != 0 && branch != 1) return fail(RT_ERR_INVALID, "branch must be 0 or 1");
  if (n < 0) return fail(RT_ERR_INVALID, "n must be >= 0");
  if (n == 0) return RT_OK;
  if ((rc = require_device_ptr(x0, "x0", false)) || (rc = require_device_ptr(dir, "dir", false)) ||
      (rc = require_device_ptr(omega, "omega", false)) || (rc = require_device_ptr(k0, "k0", false)) ||
      (rc = require_device_ptr(D_out, "D_out", true)))
    return rc;
  const rt::Params<double> P = make_params<double>(eq, kOmegaRefPerRay);
  return launch_launch(eq, disp, P, branch, x0, dir, omega, kOmegaRefPerRay, n, k0, D_out, static_cast<cudaStream_t>(cuda_stream));
}

int rt_launch_kx(const rt_equilibrium* eq, int disp, const double* x0, const double* k_guess, double omega,
                 const double* omega_rays, int64_t n, int max_iter, double tol, double* k0, double* D_out,
                 int32_t* iters_out, void* cuda_stream) {
  int rc = check_combo(eq, disp);
  if (rc) return rc;
  if (!omega_rays && (rc = check_omega(omega))) return rc;
  if (n < 0) return fail(RT_ERR_INVALID, "n must be >= 0");
  if (max_iter < 0 || max_iter > 1000) return fail(RT_ERR_INVALID, "max_iter must be in [0, 1000]");
  if (!(tol > 0.0) || !std::isfinite(tol)) return fail(RT_ERR_INVALID, "tol must be positive and finite");
  if (n == 0) return RT_OK;
  if ((rc = require_device_ptr(x0, "x0", false)) || (rc = require_device_ptr(k_guess, "k_guess", false)) ||
      (rc = require_device_ptr(omega_rays, "omega_rays", true)) || (rc = require_device_ptr(k0, "k0", false)) ||
      (rc = require_device_ptr(D_out, "D_out", true)) || (rc = require_device_ptr(iters_out, "iters_out", true, 4)))
    return rc;
  const rt::Params<double> P = make_params<double>(eq, omega_rays ? kOmegaRefPerRay : omega);
  return launch_launch_kx(eq, disp, P, x0, k_guess, omega_rays, kOmegaRefPerRay, n, max_iter, tol, k0, D_out, iters_out,
                          static_cast<cudaStream_t>(cuda_stream));
}

int rt_diagnostics(const rt_equilibrium* eq, const double* x, const double* k, double omega, const double* omega_rays,
                   int64_t n, double* out, void* cuda_stream) {
  if (!eq) return fail(RT_ERR_INVALID, "equilibrium handle is NULL");
  int rc;
  if ((rc = check_device(eq))) return rc;
  if (!omega_rays && (rc = check_omega(omega))) return rc;
  if (n < 0) return fail(RT_ERR_INVALID, "n must be >= 0");
  if (n == 0) return RT_OK;
  if ((rc = require_device_ptr(x, "x", false)) || (rc = require_device_ptr(k, "k", false)) ||
      (rc = require_device_ptr(omega_rays, "omega_rays", true)) || (rc = require_device_ptr(out, "out", false)))
    return rc;
  const double wref = omega_rays ? kOmegaRefPerRay : omega;
  const rt::Params<double> P = make_params<double>(eq, wref);
  const double inv_alpha = rt::kEps0 * rt::kMe * wref * wref / (rt::kQe * rt::kQe);   // n_e = X / alpha at w_ref
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const unsigned grid = grid_for(n, rt::AUX_BLOCK);
#define M(E)                                                                                                    \
  if (kernel_kind(eq) == (E)) {                                                                                 \
    if (omega_rays)                                                                                             \
      rt::diag_kernel<E, true><<<grid, rt::AUX_BLOCK, 0, st>>>(P, inv_alpha, x, k, omega_rays, wref, n, out);   \
    else                                                                                                        \
      rt::diag_kernel<E, false><<<grid, rt::AUX_BLOCK, 0, st>>>(P, inv_alpha, x, k, omega_rays, wref, n, out);  \
    ++g_launches;                                                                                               \
    RT_CUDA(cudaGetLastError());                                                                                \
    return RT_OK;                                                                                               \
  }
  M(rt::EQ_PARABOLIC) M(rt::EQ_LINEAR) M(rt::EQ_TOKAMAK) M(rt::EQ_TOKAMAK_POW) M(rt::EQ_GRID)
#undef M
  return fail(RT_ERR_UNSUPPORTED, "no diagnostics kernel for this equilibrium kind");
}

int rt_rhs(const rt_equilibrium* eq, int disp, int precision, const void* x, const void* k, double omega, int64_t n,
           void* D_out, void* rhs_out, int32_t* inside_out, void* cuda_stream) {
  int rc = check_combo(eq, disp);
  if (rc) return rc;
  if (precision != RT_F64 && precision != RT_F32) return fail(RT_ERR_INVALID, "unknown precision");
  if ((rc = check_omega(omega))) return rc;
  if (n < 0) return fail(RT_ERR_INVALID, "n must be >= 0");
  if (n == 0) return RT_OK;
  const size_t es = (precision == RT_F64) ? 8 : 4;
  if ((rc = require_device_ptr(x, "x", false, es)) || (rc = require_device_ptr(k, "k", false, es)) ||
      (rc = require_device_ptr(D_out, "D_out", true, es)) || (rc = require_device_ptr(rhs_out, "rhs_out", true, es)) ||
      (rc = require_device_ptr(inside_out, "inside_out", true, 4)))
    return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (precision == RT_F64)
    return launch_rhs<double>(eq, disp, make_params<double>(eq, omega), static_cast<const double*>(x),
                              static_cast<const double*>(k), n, static_cast<double*>(D_out), static_cast<double*>(rhs_out), inside_out, st);
  return launch_rhs<float>(eq, disp, make_params<float>(eq, omega), static_cast<const float*>(x), static_cast<const float*>(k), n,
                           static_cast<float*>(D_out), static_cast<float*>(rhs_out), inside_out, st);
}

int rt_reduce(int precision, const void* residual, const int32_t* status, int64_t n, double* out, void* cuda_stream) {
  if (precision != RT_F64 && precision != RT_F32) return fail(RT_ERR_INVALID, "unknown precision");
  if (n < 0) return fail(RT_ERR_INVALID, "n must be >= 0");
  int rc;
  if ((rc = require_device_ptr(out, "out", false)) ||
      (rc = require_device_ptr(residual, "residual", true, (precision == RT_F64) ? 8 : 4)) ||
      (rc = require_device_ptr(status, "status", true, 4)))
    return rc;
  return launch_reduce(precision, residual, status, n, out, static_cast<cudaStream_t>(cuda_stream));
}

int rt_fma_peak(int precision, double min_ms, double* fma_per_s, double* sm_clock_mhz) {
  // fp32: the packed shape -- the best the chip's FP32 FMA pipe delivers, so the denominator counts FMAs, not instructions
  return rt_fma_peak_shape(precision, precision == RT_F32 ? 5 : 0, 4, min_ms, fma_per_s, sm_clock_mhz);
}

int rt_fma_peak_shape(int precision, int shape, int blocks_per_sm, double min_ms, double* fma_per_s,
                      double* sm_clock_mhz) {
  if (precision != RT_F64 && precision != RT_F32) return fail(RT_ERR_INVALID, "unknown precision");
  if (shape < 0 || shape > 6 || (shape >= 5 && precision != RT_F32))
    return fail(RT_ERR_INVALID, "shape must be 0 (acc*a+acc), 1 (acc*a+b, shared a, b), 2 (acc_j*a_j+b_j), 3 (0 + MUFU), "
                                "4 (one chain), or for fp32 5 / 6 (shapes 0 / 2 with packed f32x2 accumulators)");
  if (blocks_per_sm < 1 || blocks_per_sm > 8) return fail(RT_ERR_INVALID, "blocks_per_sm must be in [1, 8]");
  if (!fma_per_s) return fail(RT_ERR_INVALID, "fma_per_s is NULL");
  if (!(min_ms > 0.0) || min_ms > 10000.0) return fail(RT_ERR_INVALID, "min_ms must be in (0, 10000]");
  int dev = 0, sms = 0;
  RT_CUDA(cudaGetDevice(&dev));
  RT_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int grid = sms * blocks_per_sm;                      // 256-thread blocks: 2 warps per scheduler each
  void* sink = nullptr;
  unsigned long long* clk = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  struct Cleanup {                                           // every early return below releases what was acquired
    void*& sink; unsigned long long*& clk; cudaEvent_t& e0; cudaEvent_t& e1;
    ~Cleanup() {
      if (e0) cudaEventDestroy(e0);
      if (e1) cudaEventDestroy(e1);
      cudaFree(sink); cudaFree(clk);
    }
  } cleanup{sink, clk, e0, e1};
  RT_CUDA(cudaMalloc(&sink, (size_t)grid * rt::FMA_BLOCK * 8));
  RT_CUDA(cudaMalloc(reinterpret_cast<void**>(&clk), 16));
  RT_CUDA(cudaEventCreate(&e0));
  RT_CUDA(cudaEventCreate(&e1));
  auto run = [&](long long iters, float* ms) -> int {
    RT_CUDA(cudaEventRecord(e0, 0));
#define RT_PEAK(T, SH, A, B) rt::fma_peak_kernel<T, SH><<<grid, rt::FMA_BLOCK>>>(static_cast<T*>(sink), iters, A, B, clk)
    if (precision == RT_F64) {
      if (shape == 0) RT_PEAK(double, 0, 1e-9, 1e-3);
      else if (shape == 1) RT_PEAK(double, 1, 0.999, 1e-3);
      else if (shape == 2) RT_PEAK(double, 2, 0.999, 1e-3);
      else if (shape == 3) RT_PEAK(double, 3, 1e-9, 1e-3);
      else RT_PEAK(double, 4, 1e-9, 1e-3);
    } else {
      if (shape == 5) rt::fma_peak_packed_kernel<5><<<grid, rt::FMA_BLOCK>>>(static_cast<float*>(sink), iters, 1e-7f, 1e-3f, clk);
      else if (shape == 6) rt::fma_peak_packed_kernel<6><<<grid, rt::FMA_BLOCK>>>(static_cast<float*>(sink), iters, 0.999f, 1e-3f, clk);
      else if (shape == 0) RT_PEAK(float, 0, 1e-7f, 1e-3f);
      else if (shape == 1) RT_PEAK(float, 1, 0.999f, 1e-3f);
      else if (shape == 2) RT_PEAK(float, 2, 0.999f, 1e-3f);
      else if (shape == 3) RT_PEAK(float, 3, 1e-7f, 1e-3f);
      else RT_PEAK(float, 4, 1e-7f, 1e-3f);
    }
#undef RT_PEAK
    ++g_launches;
    RT_CUDA(cudaGetLastError());
    RT_CUDA(cudaEventRecord(e1, 0));
    RT_CUDA(cudaEventSynchronize(e1));
    RT_CUDA(cudaEventElapsedTime(ms, e0, e1));
    return RT_OK;
  };
  float ms = 0.f;
  int rc = run(2000, &ms);                                    // warm-up + calibration
  if (!rc) rc = run(2000, &ms);
  long long iters = 2000;
  if (!rc) {
    iters = (long long)(2000.0 * min_ms / (ms > 1e-3f ? ms : 1e-3f)) + 1;
    rc = run(iters, &ms);
  }
  if (!rc) {
    const double fmas = (double)grid * rt::FMA_BLOCK * rt::FMA_CHAINS * 8.0 * (double)iters;
    *fma_per_s = fmas / (ms * 1e-3);
    if (sm_clock_mhz) {
      unsigned long long h[2] = {0, 0};
      RT_CUDA(cudaMemcpy(h, clk, 16, cudaMemcpyDeviceToHost));
      *sm_clock_mhz = h[1] ? (double)h[0] / (double)h[1] * 1e3 : 0.0;
    }
  }
  return rc;
}

int rt_math_probe(int precision, int fn, const void* x, int64_t n, void* out, void* cuda_stream) {
  if (precision != RT_F64 && precision != RT_F32) return fail(RT_ERR_INVALID, "unknown precision");
  if (fn < 0 || fn > 2) return fail(RT_ERR_INVALID, "fn must be 0 (rcp), 1 (rsqrt) or 2 (sqrt)");
  if (n < 0) return fail(RT_ERR_INVALID, "n must be >= 0");
  if (n == 0) return RT_OK;
  int rc;
  const size_t es = (precision == RT_F64) ? 8 : 4;
  if ((rc = require_device_ptr(x, "x", false, es)) || (rc = require_device_ptr(out, "out", false, es))) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const unsigned grid = grid_for(n, rt::AUX_BLOCK);
  if (precision == RT_F64)
    rt::math_probe_kernel<double><<<grid, rt::AUX_BLOCK, 0, st>>>(fn, static_cast<const double*>(x), n, static_cast<double*>(out));
  else
    rt::math_probe_kernel<float><<<grid, rt::AUX_BLOCK, 0, st>>>(fn, static_cast<const float*>(x), n, static_cast<float*>(out));
  ++g_launches;
  RT_CUDA(cudaGetLastError());
  return RT_OK;
}

}  // extern "C"
