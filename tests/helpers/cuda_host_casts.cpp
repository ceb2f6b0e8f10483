// Pin P8 helper: exposes the CUDA toolkit's HOST conversion routines (cuda_fp4.hpp /
// cuda_fp8.hpp, plain C++ when compiled with g++) so the oracle's E2M1 / E4M3 encoders can
// be checked against a library implementation they share no code with.
#include <cuda_fp4.h>
#include <cuda_fp8.h>
extern "C" unsigned char lib_e2m1(double x) {
  return (unsigned char)__nv_cvt_double_to_fp4(x, __NV_E2M1, cudaRoundNearest);
}
extern "C" unsigned char lib_e4m3(double x) {
  return (unsigned char)__nv_cvt_double_to_fp8(x, __NV_SATFINITE, __NV_E4M3);
}
