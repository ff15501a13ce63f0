// Complex helpers on float2 / double2 (interleaved re,im), shared by every kernel.
#pragma once
#include <cuda_runtime.h>

namespace gm {

template <typename T> struct cplx_of;
template <> struct cplx_of<float>  { using type = float2;  };
template <> struct cplx_of<double> { using type = double2; };
template <typename T> using cplx = typename cplx_of<T>::type;

__host__ __device__ __forceinline__ float2  mk(float x, float y)   { return make_float2(x, y); }
__host__ __device__ __forceinline__ double2 mk(double x, double y) { return make_double2(x, y); }

template <typename C> __host__ __device__ __forceinline__ C cadd(C a, C b) { return mk(a.x + b.x, a.y + b.y); }
template <typename C> __host__ __device__ __forceinline__ C csub(C a, C b) { return mk(a.x - b.x, a.y - b.y); }
template <typename C> __host__ __device__ __forceinline__ C cmul(C a, C b) {
  return mk(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
template <typename C> __host__ __device__ __forceinline__ C cmulc(C a, C b) {   // a * conj(b)
  return mk(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}
template <typename C, typename T> __host__ __device__ __forceinline__ C cscale(C a, T s) {
  return mk(a.x * s, a.y * s);
}
// multiply by +i (S > 0) or -i (S < 0)
template <int S, typename C> __host__ __device__ __forceinline__ C cmul_i(C a) {
  return S > 0 ? mk(-a.y, a.x) : mk(a.y, -a.x);
}

// Programmatic dependent launch: every kernel is launched with programmatic stream serialisation, so it may start
// while its predecessor on the stream drains.  pdl_launch_dependents() lets the successor be scheduled; pdl_wait()
// returns once every predecessor grid has completed and its memory is visible -- it precedes the kernel's first
// access (read or write) to global memory.  Both are no-ops for a kernel launched without the attribute.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_prologue() {
  pdl_launch_dependents();
  pdl_wait();
}

}  // namespace gm
