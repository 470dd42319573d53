// tfa_static.cu — tfa_face_states_static: step a2 (least-squares gradient, Venkatakrishnan limiter, face states;
// L74, L208, L232) for callers that cannot allocate device memory (CUDA graph capture, tight serving loops,
// harnesses that forbid cudaMalloc).  The kernels are the ones tfa_assemble_gradient launches; what differs is
// where their scratch lives: the least-squares coefficient vectors c_ij (two doubles per stencil entry), which
// tfa_assemble keeps in a cudaMalloc'ed workspace of the context, sit here in a file-scope __device__ array of a
// fixed maximum size, and the face states go straight to the caller's buffer.
//
// The array is one per GPU that loads the library (32 MiB each, held until the process exits) and is shared by
// every call: it keeps the last call's coefficients, every call rewrites the 2 n_stencil entries it reads (nothing
// has to start at zero), and two calls that overlap on the GPU (different streams, different threads) race on it.
#include <mutex>

#include "tfa_common.cuh"

namespace tfa {
int launch_lsq_coef(const tfa_mesh& m, double power, double* coef, cudaStream_t st);
int launch_gradient(const tfa_mesh& m, const double* state, const double* coef, double venkK, double* fown,
                    double* grad, double* phi, int32_t* flags, cudaStream_t st);
}  // namespace tfa

using namespace tfa;

namespace {

constexpr int64_t MAX_STENCIL = TFA_STATIC_MAX_STENCIL;
// scratch: coefficient pairs of up to MAX_STENCIL stencil entries; counters of the bounds-checking build
static __device__ __align__(256) double g_lsq_coef[2 * MAX_STENCIL];
static __device__ __align__(256) int32_t g_flags[4];

// In host code the names above are host-side stand-ins, not device addresses: the device address is looked up once
// per device, with that device current, and it is the looked-up pointer that goes to the kernels.
constexpr int MAX_DEVICES = 64;
struct DevicePtrs {
  double* coef = nullptr;
  int32_t* flags = nullptr;
};
DevicePtrs g_ptrs[MAX_DEVICES];
std::mutex g_ptrs_lock;

int scratch_of_current_device(DevicePtrs& out) {
  int dev = -1;
  TFA_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= MAX_DEVICES) return set_error(TFA_EINVAL, "tfa_face_states_static: device ordinal out of range");
  std::lock_guard<std::mutex> guard(g_ptrs_lock);
  if (!g_ptrs[dev].coef) {
    DevicePtrs p;
    TFA_CUDA(cudaGetSymbolAddress((void**)&p.coef, g_lsq_coef));
    TFA_CUDA(cudaGetSymbolAddress((void**)&p.flags, g_flags));
    if (!p.coef || !p.flags) return set_error(TFA_ECUDA, "tfa_face_states_static: no device address for the scratch array");
    g_ptrs[dev] = p;
  }
  out = g_ptrs[dev];
  return 0;
}

}  // namespace

extern "C" int tfa_face_states_static(const tfa_ctx* ctx, const tfa_mesh* m, const double* state, double* face_states,
                                      void* stream) {
  if (!ctx || !m) return set_error(TFA_EINVAL, "null argument");
  if (m->nc == 0) return 0;
  if (!state || !face_states) return set_error(TFA_EINVAL, "null argument");
  if (m->nst > MAX_STENCIL)
    return set_error(TFA_EINVAL, "tfa_face_states_static: the mesh has " + std::to_string(m->nst) +
                                     " stencil entries, the static scratch holds TFA_STATIC_MAX_STENCIL = " +
                                     std::to_string(MAX_STENCIL) + " (use tfa_assemble_gradient)");
  DevicePtrs p;
  TFA_TRY(scratch_of_current_device(p));
  cudaStream_t st = (cudaStream_t)stream;
  TFA_TRY(launch_lsq_coef(*m, ctx->nu.lsq_weight_power, p.coef, st));
  return launch_gradient(*m, state, p.coef, ctx->nu.venkat_K, face_states, nullptr, nullptr, p.flags, st);
}
