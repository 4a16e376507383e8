// flopcount.h -- a real-number type that counts the floating-point operations executed on it.
//
// The generated matrix elements are templates over the real type T (csrc/hg_cx.cuh), so the generator can run
// them on this type on the host and report the exact number of operations one event costs (SURVEY.md 8d:
// "algorithmic flops per event": add, sub, mul = 1; an a*b+c pair counts 2 whether or not the compiler fuses
// it; divide / reciprocal and sqrt = 1 each; negation, comparisons and copies = 0).
#pragma once
#include <math.h>

namespace hg {

struct Cnt {
  double v;
  static long long& n() {
    static long long c = 0;
    return c;
  }
  Cnt() : v(0) {}
  Cnt(double x) : v(x) {}
  Cnt(int x) : v(x) {}
  explicit operator double() const { return v; }
};
inline Cnt operator+(Cnt a, Cnt b) { ++Cnt::n(); return Cnt(a.v + b.v); }
inline Cnt operator-(Cnt a, Cnt b) { ++Cnt::n(); return Cnt(a.v - b.v); }
inline Cnt operator*(Cnt a, Cnt b) { ++Cnt::n(); return Cnt(a.v * b.v); }
inline Cnt operator-(Cnt a) { return Cnt(-a.v); }
inline Cnt& operator+=(Cnt& a, Cnt b) { ++Cnt::n(); a.v += b.v; return a; }
inline Cnt hsqrt(Cnt x) { ++Cnt::n(); return Cnt(sqrt(x.v)); }
inline Cnt hrcp(Cnt x) { ++Cnt::n(); return Cnt(1.0 / x.v); }
inline Cnt habs(Cnt x) { return Cnt(fabs(x.v)); }
inline bool hpos(Cnt x) { return x.v > 0.0; }
inline Cnt hflip(Cnt x, int flip) { return flip ? Cnt(-x.v) : x; }

}  // namespace hg
