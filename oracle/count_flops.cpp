/*
 * count_flops.cpp -- the oracle built once more with a COUNTING number type: every
 * `double` of oracle/fxoracle.c becomes a wrapper whose + - * / sqrt and comparisons bump a counter, so that one
 * fxo_hydro_advance on a small periodic tiling gives the EXACT number of floating-point operations of the method as
 * the oracle states it, per zone and RK stage.  The arithmetic is the oracle's, untouched: this file only includes it.
 *
 * TEST / MEASUREMENT INFRASTRUCTURE ONLY (like the oracle itself): built and run by oracle/count_flops.py, which writes
 * oracle/flop_counts.json; bench.py reads that file for the flop side of the roofline.
 *
 * Convention [NS]: +, -, *, /, sqrt and each comparison (min / max / floor test / branch on a value) count 1; the
 * oracle is compiled without FMA contraction, so no operation counts 2; unary minus, fabs, isfinite, copies and
 * integer index arithmetic count 0.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

struct fxo_ops { unsigned long long add, mul, div, sqrt_, cmp; };
static fxo_ops g_ops;

struct Cd {
  double v;
  Cd() = default;
  Cd(double x) : v(x) {}
  Cd(int x) : v(x) {}
  Cd(long x) : v((double)x) {}
  Cd(long long x) : v((double)x) {}
  explicit operator double() const { return v; }
  explicit operator bool() const { return v != 0.0; }
  explicit operator int() const { return (int)v; }
};
static inline Cd operator+(Cd a, Cd b) { ++g_ops.add; return Cd(a.v + b.v); }
static inline Cd operator-(Cd a, Cd b) { ++g_ops.add; return Cd(a.v - b.v); }
static inline Cd operator*(Cd a, Cd b) { ++g_ops.mul; return Cd(a.v * b.v); }
static inline Cd operator/(Cd a, Cd b) { ++g_ops.div; return Cd(a.v / b.v); }
static inline Cd operator-(Cd a) { return Cd(-a.v); }
static inline Cd &operator+=(Cd &a, Cd b) { ++g_ops.add; a.v += b.v; return a; }
static inline Cd &operator-=(Cd &a, Cd b) { ++g_ops.add; a.v -= b.v; return a; }
static inline Cd &operator*=(Cd &a, Cd b) { ++g_ops.mul; a.v *= b.v; return a; }
static inline bool operator<(Cd a, Cd b) { ++g_ops.cmp; return a.v < b.v; }
static inline bool operator>(Cd a, Cd b) { ++g_ops.cmp; return a.v > b.v; }
static inline bool operator<=(Cd a, Cd b) { ++g_ops.cmp; return a.v <= b.v; }
static inline bool operator>=(Cd a, Cd b) { ++g_ops.cmp; return a.v >= b.v; }
static inline bool operator==(Cd a, Cd b) { ++g_ops.cmp; return a.v == b.v; }
static inline bool operator!=(Cd a, Cd b) { ++g_ops.cmp; return a.v != b.v; }
static inline Cd sqrt(Cd a) { ++g_ops.sqrt_; return Cd(::sqrt(a.v)); }
static inline Cd fabs(Cd a) { return Cd(::fabs(a.v)); }
#undef isfinite
static inline bool isfinite(Cd a) { return __builtin_isfinite(a.v); }

#define double Cd
extern "C" {
#include "fxoracle.c"
}
#undef double

extern "C" void fxo_count_reset(void) { memset(&g_ops, 0, sizeof(g_ops)); }
extern "C" void fxo_count_get(unsigned long long out[5]) {
  out[0] = g_ops.add; out[1] = g_ops.mul; out[2] = g_ops.div; out[3] = g_ops.sqrt_; out[4] = g_ops.cmp;
}
