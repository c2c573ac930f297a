// mc_count.h -- host-only counting scalar for the flop model (mc_flop_model.cpp).
//
// mc::Cnt behaves like a double and counts what is done to it: fused multiply-adds, multiplications,
// additions/subtractions and special functions (rsqrt, reciprocal, division, sqrt: one each -- the Newton
// refinements the device wraps around the MUFU seeds are an implementation detail, not algorithmic work).
// Instantiating mc_math.cuh / mc_correct.cuh with T = Cnt therefore counts the operations of the formulation
// the kernels really run.  Negation, comparisons and operations between plain doubles (constants) are free.
#pragma once
#include <cmath>
#include <stdint.h>

namespace mc {

struct OpCounts { int64_t fma, mul, add, special; };
inline OpCounts& op_counts() { static thread_local OpCounts c = {0, 0, 0, 0}; return c; }

struct Cnt {
  double v;
  Cnt() : v(0.0) {}
  Cnt(double x) : v(x) {}
};
using ::fma;   // keep fma(double, double, double) visible beside the overload below
inline Cnt fma(Cnt a, Cnt b, Cnt c) { ++op_counts().fma; return Cnt(std::fma(a.v, b.v, c.v)); }
inline Cnt operator*(Cnt a, Cnt b) { ++op_counts().mul; return Cnt(a.v * b.v); }
inline Cnt operator+(Cnt a, Cnt b) { ++op_counts().add; return Cnt(a.v + b.v); }
inline Cnt operator-(Cnt a, Cnt b) { ++op_counts().add; return Cnt(a.v - b.v); }
inline Cnt operator-(Cnt a) { return Cnt(-a.v); }
inline Cnt& operator*=(Cnt& a, Cnt b) { a = a * b; return a; }
inline Cnt& operator+=(Cnt& a, Cnt b) { a = a + b; return a; }
inline Cnt& operator-=(Cnt& a, Cnt b) { a = a - b; return a; }
inline bool operator<(Cnt a, Cnt b) { return a.v < b.v; }
inline bool operator>(Cnt a, Cnt b) { return a.v > b.v; }
inline bool operator<=(Cnt a, Cnt b) { return a.v <= b.v; }
inline bool operator>=(Cnt a, Cnt b) { return a.v >= b.v; }
inline bool operator!=(Cnt a, Cnt b) { return a.v != b.v; }
inline bool operator==(Cnt a, Cnt b) { return a.v == b.v; }
inline Cnt rsqrt_pos(Cnt x) { ++op_counts().special; return Cnt(1.0 / std::sqrt(x.v)); }
inline Cnt rcp_nz(Cnt x) { ++op_counts().special; return Cnt(1.0 / x.v); }
inline Cnt sqrt_pos(Cnt x) { ++op_counts().special; return Cnt(std::sqrt(x.v)); }
inline Cnt div_(Cnt a, Cnt b) { ++op_counts().special; return Cnt(a.v / b.v); }
inline Cnt div_exact(Cnt a, Cnt b) { ++op_counts().special; return Cnt(a.v / b.v); }
inline Cnt log10_(Cnt x) { return Cnt(std::log10(x.v)); }   // the logarithm of the FLI is bookkeeping, not counted
inline Cnt abs_(Cnt x) { return Cnt(std::fabs(x.v)); }
inline bool is_finite(Cnt x) { return std::isfinite(x.v); }
inline bool warp_any(bool b) { return b; }

}  // namespace mc
