// counted_real.h -- an operation-counting scalar for the CPU oracle (TEST INFRASTRUCTURE).
// Build oracle/hzo.cpp with  -DHZO_CUSTOM_REAL -DHZO_REAL=Counted -include counted_real.h  (no OpenMP):
// every +, -, *, /, sqrt, comparison and abs/min/max on `real` is tallied, which gives the algorithmic
// operation count per zone and substep that DESIGN.md section 5 uses for the ALU roofline.
#pragma once
#include <cmath>
struct OpCounts { long long add, mul, div, sqrt, cmp, absminmax; };
inline OpCounts& hzo_ops() { static OpCounts c = {0, 0, 0, 0, 0, 0}; return c; }
struct Counted {
  double v;
  Counted() : v(0) {}
  Counted(double x) : v(x) {}
  Counted(int x) : v(x) {}
  explicit operator double() const { return v; }
};
inline Counted operator+(Counted a, Counted b) { hzo_ops().add++; return Counted(a.v + b.v); }
inline Counted operator-(Counted a, Counted b) { hzo_ops().add++; return Counted(a.v - b.v); }
inline Counted operator*(Counted a, Counted b) { hzo_ops().mul++; return Counted(a.v * b.v); }
inline Counted operator/(Counted a, Counted b) { hzo_ops().div++; return Counted(a.v / b.v); }
inline Counted operator-(Counted a) { return Counted(-a.v); }
inline Counted& operator+=(Counted& a, Counted b) { hzo_ops().add++; a.v += b.v; return a; }
inline Counted& operator-=(Counted& a, Counted b) { hzo_ops().add++; a.v -= b.v; return a; }
inline Counted& operator*=(Counted& a, Counted b) { hzo_ops().mul++; a.v *= b.v; return a; }
inline Counted& operator/=(Counted& a, Counted b) { hzo_ops().div++; a.v /= b.v; return a; }
#define HZO_CMP(op) inline bool operator op(Counted a, Counted b) { hzo_ops().cmp++; return a.v op b.v; }
HZO_CMP(<) HZO_CMP(>) HZO_CMP(<=) HZO_CMP(>=) HZO_CMP(==) HZO_CMP(!=)
#undef HZO_CMP
typedef Counted real_t_for_oracle;
static inline Counted r_sqrt(Counted x) { hzo_ops().sqrt++; return Counted(std::sqrt(x.v)); }
static inline Counted r_abs(Counted x) { hzo_ops().absminmax++; return Counted(std::fabs(x.v)); }
static inline Counted r_min(Counted a, Counted b) { hzo_ops().absminmax++; return a.v < b.v ? a : b; }
static inline Counted r_max(Counted a, Counted b) { hzo_ops().absminmax++; return a.v > b.v ? a : b; }
static inline bool r_finite(Counted x) { return std::isfinite(x.v); }
static inline double r_val(Counted x) { return x.v; }
extern "C" __attribute__((used, visibility("default"))) inline void hzo_opcount_read(long long* out6, int reset) {
  OpCounts& c = hzo_ops();
  out6[0] = c.add; out6[1] = c.mul; out6[2] = c.div; out6[3] = c.sqrt; out6[4] = c.cmp; out6[5] = c.absminmax;
  if (reset) c = OpCounts{0, 0, 0, 0, 0, 0};
}
