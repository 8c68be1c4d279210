// cuda_rt_stub.hpp -- the few CUDA runtime calls csrc/chemora.cu makes, on host memory, so that the library's HOST
// code (handle, layout, stage plans, runtime sweep and its guard, timing pool, error-word plumbing) compiles with g++
// next to the emulated kernels (cta_emu.hpp) and the real C ABI can be exercised on a box without a GPU.
// Test infrastructure only: built by tests/test_abi_emulated.py into a library of its own, never loaded by the package.
//   "device" memory = 256-byte aligned host memory; copies and memsets are synchronous; one "device", no streams;
//   events carry a steady_clock time stamp.
#pragma once
#include <chrono>
#include <cstdlib>
#include <cstring>

enum cudaMemcpyKind { cudaMemcpyHostToHost = 0, cudaMemcpyHostToDevice = 1, cudaMemcpyDeviceToHost = 2, cudaMemcpyDeviceToDevice = 3 };
enum { cudaDevAttrMultiProcessorCount = 16 };
enum { cudaErrorMemoryAllocation = 2 };   // cudaSuccess, cudaErrorInvalidValue: cta_emu.hpp

struct CudaEventStub { std::chrono::steady_clock::time_point t; };
typedef CudaEventStub* cudaEvent_t;

inline cudaError_t cudaGetDeviceCount(int* n) { *n = 1; return cudaSuccess; }
inline cudaError_t cudaGetDevice(int* d) { *d = 0; return cudaSuccess; }
inline cudaError_t cudaDeviceGetAttribute(int* v, int, int) { *v = 4; return cudaSuccess; }   // 4 "SMs": grids stay small
inline cudaError_t cudaGetLastError() { return cudaSuccess; }
inline const char* cudaGetErrorString(cudaError_t e) { return e == cudaSuccess ? "no error" : e == cudaErrorInvalidValue ? "invalid argument" : "error (emulated runtime)"; }

inline cudaError_t cudaMalloc(void** p, size_t bytes) {
  *p = aligned_alloc(256, (bytes + 255) / 256 * 256);
  return *p ? (cudaError_t)cudaSuccess : (cudaError_t)cudaErrorMemoryAllocation;
}
inline cudaError_t cudaFree(void* p) { free(p); return cudaSuccess; }
inline cudaError_t cudaMemsetAsync(void* p, int v, size_t n, cudaStream_t) { memset(p, v, n); return cudaSuccess; }
inline cudaError_t cudaMemcpyAsync(void* d, const void* s, size_t n, cudaMemcpyKind, cudaStream_t) { memmove(d, s, n); return cudaSuccess; }
inline cudaError_t cudaStreamSynchronize(cudaStream_t) { return cudaSuccess; }

inline cudaError_t cudaEventCreate(cudaEvent_t* e) { *e = new CudaEventStub(); return cudaSuccess; }
inline cudaError_t cudaEventDestroy(cudaEvent_t e) { delete e; return cudaSuccess; }
inline cudaError_t cudaEventRecord(cudaEvent_t e, cudaStream_t) { e->t = std::chrono::steady_clock::now(); return cudaSuccess; }
inline cudaError_t cudaEventSynchronize(cudaEvent_t) { return cudaSuccess; }
inline cudaError_t cudaEventElapsedTime(float* ms, cudaEvent_t a, cudaEvent_t b) {
  *ms = std::chrono::duration<float, std::milli>(b->t - a->t).count();
  return cudaSuccess;
}
