// flopcount.h -- counting scalar for the INSTRUMENTED build of the oracle (TEST / MEASUREMENT INFRASTRUCTURE).
//
// SURVEY.md Sec. 8(d) asks for the algorithmic flop count of one zone-cycle from "a counting double wrapper" in the
// oracle, because the iteration counts of the recovery are data dependent.  oracle/count_flops.py builds
// rgrmhd_oracle.cpp with -DORACLE_COUNT_FLOPS; that build includes this header and then `#define double cdouble`, so
// every arithmetic operation of the oracle's own code is tallied (add/sub, mul, div, sqrt each 1 flop: a fused
// multiply-add would therefore count 2, a division or square root 1, as the roofline convention of DESIGN.md Sec. 7.5
// states), per REGION of the step (reconstruction, Riemann solve, sources, recovery, ...).  Comparisons, fabs, min/max
// and copies are free.  Results are identical to the plain build (the wrapper only forwards to double).
#pragma once
#include <cmath>
#include <limits>

namespace flopcount {
enum Region { R_OTHER = 0, R_RECON, R_RIEMANN, R_DIVERGENCE, R_SOURCES, R_C2P_SETUP, R_C2P_EVAL, R_COMBINE, R_P2C, R_COUNT };
enum Op { OP_ADD = 0, OP_MUL, OP_DIV, OP_SQRT, OP_COUNT };
extern long long counts[R_COUNT][OP_COUNT];
extern long long calls[R_COUNT];      // how many times a region was entered
extern int region;
struct Scope {                         // RAII region marker
  int prev;
  explicit Scope(int r) : prev(region) { region = r; ++calls[r]; }
  ~Scope() { region = prev; }
};
inline void tick(int op) { ++counts[region][op]; }
}  // namespace flopcount

struct cdouble {
  double v;
  cdouble() = default;
  cdouble(double x) : v(x) {}          // implicit: literals and ints mix freely
  explicit operator double() const { return v; }
  explicit operator int() const { return (int)v; }
  explicit operator long() const { return (long)v; }
  cdouble& operator+=(cdouble o) { flopcount::tick(flopcount::OP_ADD); v += o.v; return *this; }
  cdouble& operator-=(cdouble o) { flopcount::tick(flopcount::OP_ADD); v -= o.v; return *this; }
  cdouble& operator*=(cdouble o) { flopcount::tick(flopcount::OP_MUL); v *= o.v; return *this; }
  cdouble& operator/=(cdouble o) { flopcount::tick(flopcount::OP_DIV); v /= o.v; return *this; }
};
inline cdouble operator+(cdouble a, cdouble b) { flopcount::tick(flopcount::OP_ADD); return cdouble(a.v + b.v); }
inline cdouble operator-(cdouble a, cdouble b) { flopcount::tick(flopcount::OP_ADD); return cdouble(a.v - b.v); }
inline cdouble operator*(cdouble a, cdouble b) { flopcount::tick(flopcount::OP_MUL); return cdouble(a.v * b.v); }
inline cdouble operator/(cdouble a, cdouble b) { flopcount::tick(flopcount::OP_DIV); return cdouble(a.v / b.v); }
inline cdouble operator-(cdouble a) { return cdouble(-a.v); }
inline cdouble operator+(cdouble a) { return a; }
#define FLOPCOUNT_MIXED(op)                                                     \
  inline cdouble operator op(cdouble a, double b) { return a op cdouble(b); }  \
  inline cdouble operator op(double a, cdouble b) { return cdouble(a) op b; }  \
  inline cdouble operator op(cdouble a, int b) { return a op cdouble((double)b); } \
  inline cdouble operator op(int a, cdouble b) { return cdouble((double)a) op b; }
FLOPCOUNT_MIXED(+) FLOPCOUNT_MIXED(-) FLOPCOUNT_MIXED(*) FLOPCOUNT_MIXED(/)
#undef FLOPCOUNT_MIXED
#define FLOPCOUNT_CMP(op)                                                      \
  inline bool operator op(cdouble a, cdouble b) { return a.v op b.v; }         \
  inline bool operator op(cdouble a, double b) { return a.v op b; }            \
  inline bool operator op(double a, cdouble b) { return a op b.v; }
FLOPCOUNT_CMP(<) FLOPCOUNT_CMP(>) FLOPCOUNT_CMP(<=) FLOPCOUNT_CMP(>=) FLOPCOUNT_CMP(==) FLOPCOUNT_CMP(!=)
#undef FLOPCOUNT_CMP
inline bool operator!(cdouble a) { return !a.v; }

namespace std {   // the oracle calls these with the std:: prefix
inline cdouble sqrt(cdouble a) { flopcount::tick(flopcount::OP_SQRT); return cdouble(std::sqrt(a.v)); }
inline cdouble fabs(cdouble a) { return cdouble(std::fabs(a.v)); }
inline bool isfinite(cdouble a) { return std::isfinite(a.v); }
inline cdouble pow(cdouble a, cdouble b) { flopcount::tick(flopcount::OP_MUL); return cdouble(std::pow(a.v, b.v)); }
inline long lround(cdouble a) { return std::lround(a.v); }
inline cdouble max(cdouble a, double b) { return a.v < b ? cdouble(b) : a; }
inline cdouble max(double a, cdouble b) { return a < b.v ? b : cdouble(a); }
inline cdouble min(cdouble a, double b) { return b < a.v ? cdouble(b) : a; }
inline cdouble min(double a, cdouble b) { return b.v < a ? b : cdouble(a); }
template <> struct numeric_limits<cdouble> {
  static cdouble epsilon() { return cdouble(numeric_limits<double>::epsilon()); }
};
}  // namespace std
