// hg_cx.cuh -- complex numbers, real 4-momenta and small helpers for the device function library.
//
// Role of List 2 `cmplx.h`: the paper uses struct {double re, im} aligned 8 with
// overloaded operators.  Here the real type T is a template parameter (double, float, or the host-side
// flop-counting type of gen/flopcount), everything lives in registers, and every routine is
// __host__ __device__ so the generator can run the generated code on a counting type at build time.
#pragma once

#if defined(__CUDACC__)
#define HG_HD __host__ __device__ __forceinline__
#else
#define HG_HD inline
#endif

#include <math.h>

namespace hg {

// ---- scalar math wrappers (overloaded for the counting type in gen/flopcount.h) ----
HG_HD double hsqrt(double x) { return sqrt(x); }
HG_HD float hsqrt(float x) { return sqrtf(x); }
HG_HD double hrcp(double x) { return 1.0 / x; }
HG_HD float hrcp(float x) { return 1.0f / x; }
HG_HD double habs(double x) { return fabs(x); }
HG_HD float habs(float x) { return fabsf(x); }
HG_HD bool hpos(double x) { return x > 0.0; }  // the only comparisons the library makes are "x > 0"
HG_HD bool hpos(float x) { return x > 0.0f; }
// x or -x under a run-time flag (the helicity -1 polarisation vector from the staged +1 one): on the device one
// integer XOR of the sign bit instead of a negation and a select per word (the flag is loop-invariant, the mask too)
HG_HD double hflip(double x, int flip) {
#if defined(__CUDA_ARCH__)
  return __hiloint2double(__double2hiint(x) ^ (flip ? (int)0x80000000 : 0), __double2loint(x));
#else
  return flip ? -x : x;
#endif
}
HG_HD float hflip(float x, int flip) {
#if defined(__CUDA_ARCH__)
  return __int_as_float(__float_as_int(x) ^ (flip ? (int)0x80000000 : 0));
#else
  return flip ? -x : x;
#endif
}

template <class T>
struct cx {
  T re, im;
};

template <class T>
HG_HD cx<T> mk(T re, T im) {
  cx<T> r;
  r.re = re;
  r.im = im;
  return r;
}
template <class T>
HG_HD cx<T> czero() {
  return mk<T>(T(0), T(0));
}
template <class T>
HG_HD cx<T> operator+(cx<T> a, cx<T> b) {
  return mk<T>(a.re + b.re, a.im + b.im);
}
template <class T>
HG_HD cx<T> operator-(cx<T> a, cx<T> b) {
  return mk<T>(a.re - b.re, a.im - b.im);
}
template <class T>
HG_HD cx<T> operator-(cx<T> a) {
  return mk<T>(-a.re, -a.im);
}
template <class T>
HG_HD cx<T> operator*(cx<T> a, cx<T> b) {
  return mk<T>(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re);
}
template <class T>
HG_HD cx<T> operator*(T a, cx<T> b) {
  return mk<T>(a * b.re, a * b.im);
}
template <class T>
HG_HD cx<T> operator*(cx<T> a, T b) {
  return mk<T>(a.re * b, a.im * b);
}
template <class T>
HG_HD cx<T> conj(cx<T> a) {
  return mk<T>(a.re, -a.im);
}
// a + b*c
template <class T>
HG_HD cx<T> cfma(cx<T> b, cx<T> c, cx<T> a) {
  return mk<T>(a.re + b.re * c.re - b.im * c.im, a.im + b.re * c.im + b.im * c.re);
}
// i*a
template <class T>
HG_HD cx<T> times_i(cx<T> a) {
  return mk<T>(-a.im, a.re);
}
template <class T>
HG_HD T norm2(cx<T> a) {
  return a.re * a.re + a.im * a.im;
}
// 1/(x + i y)
template <class T>
HG_HD cx<T> crcp(T x, T y) {
  T s = hrcp(x * x + y * y);
  return mk<T>(x * s, -(y * s));
}

// ---- real 4-vector with upper index (E, px, py, pz) ----
template <class T>
struct Mom {
  T e, x, y, z;
};
template <class T>
HG_HD Mom<T> mkmom(T e, T x, T y, T z) {
  Mom<T> r;
  r.e = e;
  r.x = x;
  r.y = y;
  r.z = z;
  return r;
}
template <class T>
HG_HD Mom<T> operator+(Mom<T> a, Mom<T> b) {
  return mkmom<T>(a.e + b.e, a.x + b.x, a.y + b.y, a.z + b.z);
}
template <class T>
HG_HD Mom<T> operator-(Mom<T> a, Mom<T> b) {
  return mkmom<T>(a.e - b.e, a.x - b.x, a.y - b.y, a.z - b.z);
}
template <class T>
HG_HD Mom<T> operator-(Mom<T> a) {
  return mkmom<T>(-a.e, -a.x, -a.y, -a.z);
}
template <class T>
HG_HD T mdot(Mom<T> a, Mom<T> b) {
  return a.e * b.e - a.x * b.x - a.y * b.y - a.z * b.z;
}

// Invariant of a pair of MASSLESS momenta without cancellation for collinear pairs:
//   2 a.b = 2 Ea Eb (1 - cos) = Ea Eb |a^ - b^|^2 ,  a^ = a/Ea.   unit0 keeps E and stores the unit 3-vector.
template <class T>
HG_HD Mom<T> unit0(const Mom<T>& p) {
  T r = hrcp(p.e);
  return mkmom<T>(p.e, p.x * r, p.y * r, p.z * r);
}
template <class T>
HG_HD T two_dot0(const Mom<T>& a, const Mom<T>& b) {
  T dx = a.x - b.x, dy = a.y - b.y, dz = a.z - b.z;
  return a.e * b.e * (dx * dx + dy * dy + dz * dz);
}

// ---- wavefunctions: 4 complex components.  Momenta are NOT carried in the wavefunction (the paper's
// cmplx w[6] keeps them in w[4], w[5]): they are helicity independent, so the
// generator keeps them as separate Mom<T> values computed once per event. ----
template <class T>
struct Vc {  // Lorentz vector, upper index
  cx<T> c[4];
};
template <class T>
struct Sp {  // Dirac spinor in the chiral representation: slots A = c[0],c[1]; slots B = c[2],c[3]
  cx<T> c[4];
};

// sums of wavefunctions (merged currents of the generator)
template <class T>
HG_HD Vc<T> operator+(const Vc<T>& a, const Vc<T>& b) {
  Vc<T> r;
  for (int i = 0; i < 4; ++i) r.c[i] = a.c[i] + b.c[i];
  return r;
}
template <class T>
HG_HD Vc<T> operator-(const Vc<T>& a, const Vc<T>& b) {
  Vc<T> r;
  for (int i = 0; i < 4; ++i) r.c[i] = a.c[i] - b.c[i];
  return r;
}
template <class T>
HG_HD Vc<T> operator-(const Vc<T>& a) {
  Vc<T> r;
  for (int i = 0; i < 4; ++i) r.c[i] = -a.c[i];
  return r;
}
template <class T>
HG_HD Sp<T> operator+(const Sp<T>& a, const Sp<T>& b) {
  Sp<T> r;
  for (int i = 0; i < 4; ++i) r.c[i] = a.c[i] + b.c[i];
  return r;
}
template <class T>
HG_HD Sp<T> operator-(const Sp<T>& a, const Sp<T>& b) {
  Sp<T> r;
  for (int i = 0; i < 4; ++i) r.c[i] = a.c[i] - b.c[i];
  return r;
}
template <class T>
HG_HD Sp<T> operator-(const Sp<T>& a) {
  Sp<T> r;
  for (int i = 0; i < 4; ++i) r.c[i] = -a.c[i];
  return r;
}

// Minkowski products (no complex conjugation)
template <class T>
HG_HD cx<T> vdot(const Vc<T>& a, const Vc<T>& b) {
  cx<T> r = a.c[0] * b.c[0];
  r = r - a.c[1] * b.c[1];
  r = r - a.c[2] * b.c[2];
  r = r - a.c[3] * b.c[3];
  return r;
}
template <class T>
HG_HD cx<T> vdot(const Mom<T>& k, const Vc<T>& a) {
  return mk<T>(k.e * a.c[0].re - k.x * a.c[1].re - k.y * a.c[2].re - k.z * a.c[3].re,
               k.e * a.c[0].im - k.x * a.c[1].im - k.y * a.c[2].im - k.z * a.c[3].im);
}

// Slot / coupling masks: compile-time sparsity of spinors and chiral couplings (see hg_helas.cuh).
enum : int { SLOT_A = 1, SLOT_B = 2, SLOT_AB = 3 };
enum : int { CPL_L = 1, CPL_R = 2, CPL_LR = 3 };

}  // namespace hg
