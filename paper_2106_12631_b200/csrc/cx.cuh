// cx.cuh — minimal complex arithmetic for the sm_100a kernels ("thin wrapper" complex
// type).  Two scalars, everything inlined; products are written as FMA chains so that ptxas emits
// DFMA/FFMA rather than separate multiplies and adds.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

#define MG_HD __host__ __device__ __forceinline__

namespace mg {

template <class T> MG_HD T fma_(T a, T b, T c);
template <> MG_HD double fma_<double>(double a, double b, double c) { return fma(a, b, c); }
template <> MG_HD float fma_<float>(float a, float b, float c) { return fmaf(a, b, c); }
template <class T> MG_HD T sqrt_(T a);
template <> MG_HD double sqrt_<double>(double a) { return sqrt(a); }
template <> MG_HD float sqrt_<float>(float a) { return sqrtf(a); }
// 1/sqrt(a) in one step (one MUFU.RSQ seed + Newton instead of a square root followed by a division)
template <class T> MG_HD T rsqrt_(T a);
#ifdef __CUDA_ARCH__
template <> MG_HD double rsqrt_<double>(double a) { return rsqrt(a); }
template <> MG_HD float rsqrt_<float>(float a) { return rsqrtf(a); }
#else
template <> MG_HD double rsqrt_<double>(double a) { return 1.0 / sqrt(a); }
template <> MG_HD float rsqrt_<float>(float a) { return 1.0f / sqrtf(a); }
#endif
template <class T> MG_HD T abs_(T a) { return a < (T)0 ? -a : a; }

template <class T> struct cx {
  T re, im;
  MG_HD cx() {}
  MG_HD cx(T r, T i) : re(r), im(i) {}
};

template <class T> MG_HD cx<T> operator+(cx<T> a, cx<T> b) { return cx<T>(a.re + b.re, a.im + b.im); }
template <class T> MG_HD cx<T> operator-(cx<T> a, cx<T> b) { return cx<T>(a.re - b.re, a.im - b.im); }
template <class T> MG_HD cx<T> operator-(cx<T> a) { return cx<T>(-a.re, -a.im); }
// a*b : 2 mul + 2 fma
template <class T> MG_HD cx<T> operator*(cx<T> a, cx<T> b) {
  return cx<T>(fma_<T>(-a.im, b.im, a.re * b.re), fma_<T>(a.im, b.re, a.re * b.im));
}
template <class T> MG_HD cx<T> operator*(T s, cx<T> a) { return cx<T>(s * a.re, s * a.im); }
template <class T> MG_HD cx<T> operator*(cx<T> a, T s) { return cx<T>(s * a.re, s * a.im); }
// acc + a*b : 4 fma
template <class T> MG_HD cx<T> cfma(cx<T> a, cx<T> b, cx<T> acc) {
  T re = fma_<T>(a.re, b.re, acc.re);
  T im = fma_<T>(a.re, b.im, acc.im);
  return cx<T>(fma_<T>(-a.im, b.im, re), fma_<T>(a.im, b.re, im));
}
// acc - a*b : 4 fma
template <class T> MG_HD cx<T> cfms(cx<T> a, cx<T> b, cx<T> acc) {
  T re = fma_<T>(-a.re, b.re, acc.re);
  T im = fma_<T>(-a.re, b.im, acc.im);
  return cx<T>(fma_<T>(a.im, b.im, re), fma_<T>(-a.im, b.re, im));
}
// acc + s*a (s real): 2 fma
template <class T> MG_HD cx<T> rfma(T s, cx<T> a, cx<T> acc) {
  return cx<T>(fma_<T>(s, a.re, acc.re), fma_<T>(s, a.im, acc.im));
}
template <class T> MG_HD cx<T> conj_(cx<T> a) { return cx<T>(a.re, -a.im); }
template <class T> MG_HD cx<T> times_i(cx<T> a) { return cx<T>(-a.im, a.re); }
template <class T> MG_HD cx<T> times_mi(cx<T> a) { return cx<T>(a.im, -a.re); }
template <class T> MG_HD T norm2(cx<T> a) { return fma_<T>(a.re, a.re, a.im * a.im); }

}  // namespace mg
