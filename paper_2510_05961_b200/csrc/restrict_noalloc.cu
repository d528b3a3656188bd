// restrict_noalloc.cu -- msm_restrict_noalloc: the separable restriction Q^{l+1} = I_l^{l+1} Q^l
// (Eq. 19 line 1, one axis at a time) for callers that cannot allocate device memory
// (code under CUDA-graph capture, serving loops, harnesses that forbid cudaMalloc).
//
// The plan path keeps the two intermediate arrays of the three axis passes (after x: coarse in x,
// fine in y and z; after y: coarse in x and y, fine in z) in plan-owned buffers that
// msm_plan_create allocates. Here they live in ONE file-scope device array of
// MSM_NOALLOC_SCRATCH_BYTES that every GPU which loads the library holds until the process exits.
// The entry point calls no cudaMalloc / cudaFree and no allocating library routine; its only
// set-up is cudaGetSymbolAddress, once per device, which returns the address of storage that
// already exists.
//
// Sharing rules. Every call on a device uses the same array: two calls that overlap on the GPU
// (different streams without an event between them) race on it. Calls on one stream are ordered
// and safe. The array keeps the last call's contents; nothing has to start at zero, because each
// pass writes every element of its output region before the next pass reads it (one thread per
// output element, no accumulation into memory), so no clearing launch is needed.
#include <cuda_runtime.h>

#include <mutex>

#include "../../include/msm.h"
#include "gridops.cuh"

namespace {

using namespace msm;

// file-scope scratch: the x-pass output at offset 0, the y-pass output behind it (256-byte aligned)
static __device__ __align__(256) unsigned char g_noalloc_scratch[MSM_NOALLOC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;
std::mutex g_addr_mutex;
void* g_scratch_addr[kMaxDevices] = {};   // device address of g_noalloc_scratch per device ordinal

// In host code g_noalloc_scratch is a host-side stand-in, not a device address: look the device
// address up once per device, with that device current.
msm_status_t scratch_address(int device, unsigned char** out) {
  std::lock_guard<std::mutex> lock(g_addr_mutex);
  if (!g_scratch_addr[device]) {
    void* ptr = nullptr;
    if (cudaGetSymbolAddress(&ptr, g_noalloc_scratch) != cudaSuccess || !ptr) {
      cudaGetLastError();
      return MSM_ERR_CUDA;
    }
    g_scratch_addr[device] = ptr;
  }
  *out = (unsigned char*)g_scratch_addr[device];
  return MSM_OK;
}

struct RestoreDevice {
  int prev = -1;
  ~RestoreDevice() { if (prev >= 0) cudaSetDevice(prev); }
};

template <typename T>
msm_status_t run(int p, const int* fd, const int* flo, const int* cd, const int* clo, const int* periodic,
                 const T* fine, T* coarse, unsigned char* scratch, size_t off_b, cudaStream_t st) {
  AxisTaps<T> J;                           // J_n = 2^(1-p) binom(p, n + p/2) (reading J1)
  J.n = p + 1;
  double b = 1.0;
  for (int k = 0; k <= p; ++k) {
    J.c[k] = (T)(b / (double)(1u << (p - 1)));
    b = b * (p - k) / (k + 1.0);
  }
  T* after_x = (T*)scratch;
  T* after_y = (T*)(scratch + off_b);
  int din[3] = {fd[0], fd[1], fd[2]};
  const T* src = fine;
  for (int ax = 0; ax < 3; ++ax) {
    AxisDims d;
    for (int k = 0; k < 3; ++k) { d.in[k] = din[k]; d.out[k] = din[k]; }
    d.out[ax] = cd[ax];
    d.axis = ax;
    d.periodic = periodic[ax] ? 1 : 0;
    T* dst = ax == 0 ? after_x : (ax == 1 ? after_y : coarse);
    if (ax == 0) k_restrict_axis<T, 0><<<axis_grid(d), axis_block(), 0, st>>>(d, flo[ax], clo[ax], J, src, dst);
    else if (ax == 1) k_restrict_axis<T, 1><<<axis_grid(d), axis_block(), 0, st>>>(d, flo[ax], clo[ax], J, src, dst);
    else k_restrict_axis<T, 2><<<axis_grid(d), axis_block(), 0, st>>>(d, flo[ax], clo[ax], J, src, dst);
    if (cudaGetLastError() != cudaSuccess) return MSM_ERR_CUDA;
    src = dst;
    din[ax] = cd[ax];
  }
  return MSM_OK;
}

}  // namespace

extern "C" msm_status_t msm_restrict_noalloc(int device, int precision, int p, const int* fine_dims,
                                             const int* fine_lo, const int* coarse_dims, const int* coarse_lo,
                                             const int* periodic, const void* d_fine, void* d_coarse,
                                             void* cuda_stream) {
  if (!fine_dims || !fine_lo || !coarse_dims || !coarse_lo || !periodic || !d_fine || !d_coarse)
    return MSM_ERR_INVALID_ARG;
  if (device < 0 || device >= kMaxDevices) return MSM_ERR_INVALID_ARG;
  if (precision != MSM_FP64 && precision != MSM_FP32) return MSM_ERR_INVALID_ARG;
  if (p != 4 && p != 6 && p != 8) return MSM_ERR_INVALID_ARG;
  for (int ax = 0; ax < 3; ++ax)
    if (fine_dims[ax] < 1 || coarse_dims[ax] < 1 || coarse_dims[ax] > fine_dims[ax]) return MSM_ERR_INVALID_ARG;
  const size_t esz = precision == MSM_FP32 ? sizeof(float) : sizeof(double);
  const size_t fine_pts = (size_t)fine_dims[0] * fine_dims[1] * fine_dims[2];
  if (fine_pts >= ((size_t)1 << 31)) return MSM_ERR_SCRATCH_LIMIT;   // (32-bit index maths; far above the limit below)
  // scratch: after x (cx, fy, fz), after y (cx, cy, fz)
  const size_t bytes_a = (size_t)coarse_dims[0] * fine_dims[1] * fine_dims[2] * esz;
  const size_t bytes_b = (size_t)coarse_dims[0] * coarse_dims[1] * fine_dims[2] * esz;
  const size_t off_b = (bytes_a + 255) / 256 * 256;
  if (off_b + bytes_b > (size_t)MSM_NOALLOC_SCRATCH_BYTES) return MSM_ERR_SCRATCH_LIMIT;

  RestoreDevice guard;
  if (cudaGetDevice(&guard.prev) != cudaSuccess) guard.prev = -1;
  if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return MSM_ERR_CUDA; }
  unsigned char* scratch = nullptr;
  const msm_status_t s = scratch_address(device, &scratch);
  if (s != MSM_OK) return s;
  const cudaStream_t st = (cudaStream_t)cuda_stream;
  if (precision == MSM_FP32)
    return run<float>(p, fine_dims, fine_lo, coarse_dims, coarse_lo, periodic, (const float*)d_fine, (float*)d_coarse,
                      scratch, off_b, st);
  return run<double>(p, fine_dims, fine_lo, coarse_dims, coarse_lo, periodic, (const double*)d_fine, (double*)d_coarse,
                     scratch, off_b, st);
}
