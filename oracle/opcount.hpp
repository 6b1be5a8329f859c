// opcount.hpp -- an operation-counting scalar for the CPU oracle (TEST INFRASTRUCTURE, see dock_oracle.h).
// dock_oracle_count.cpp compiles the UNCHANGED dock_oracle.c with `double` replaced by this type, so that the
// algorithmic floating-point work of one score+gradient evaluation (SURVEY.md 8(d) "the final flop count is taken
// from the oracle run with an operation-counting scalar type") is counted on the oracle's own statements:
// one per add / sub / mul / div / compare / sqrt / exp / sin / cos / floor / fabs / fmin, nothing fused.
// Counters are plain globals: call the single-threaded entry points (orc_eval, orc_pair ...) only.
#pragma once
#include <math.h>
#include <stdint.h>

enum { OC_ADD, OC_MUL, OC_DIV, OC_CMP, OC_SQRT, OC_EXP, OC_TRIG, OC_MISC, OC_N };
extern "C" uint64_t g_opcount[OC_N];

struct cdouble {
    double v;
    cdouble() = default;
    cdouble(double x) : v(x) {}
    explicit operator double() const { return v; }
    explicit operator float() const { return (float)v; }
    explicit operator int() const { return (int)v; }
    explicit operator long() const { return (long)v; }
    explicit operator long long() const { return (long long)v; }
    explicit operator unsigned() const { return (unsigned)v; }
    cdouble &operator+=(cdouble o) { ++g_opcount[OC_ADD]; v += o.v; return *this; }
    cdouble &operator-=(cdouble o) { ++g_opcount[OC_ADD]; v -= o.v; return *this; }
    cdouble &operator*=(cdouble o) { ++g_opcount[OC_MUL]; v *= o.v; return *this; }
    cdouble &operator/=(cdouble o) { ++g_opcount[OC_DIV]; v /= o.v; return *this; }
    cdouble operator-() const { return cdouble(-v); }          // a sign flip is not counted
};
static_assert(sizeof(cdouble) == sizeof(double), "cdouble must have the layout of double (the ctypes binding relies on it)");

inline cdouble operator+(cdouble a, cdouble b) { ++g_opcount[OC_ADD]; return cdouble(a.v + b.v); }
inline cdouble operator-(cdouble a, cdouble b) { ++g_opcount[OC_ADD]; return cdouble(a.v - b.v); }
inline cdouble operator*(cdouble a, cdouble b) { ++g_opcount[OC_MUL]; return cdouble(a.v * b.v); }
inline cdouble operator/(cdouble a, cdouble b) { ++g_opcount[OC_DIV]; return cdouble(a.v / b.v); }
inline bool operator<(cdouble a, cdouble b) { ++g_opcount[OC_CMP]; return a.v < b.v; }
inline bool operator>(cdouble a, cdouble b) { ++g_opcount[OC_CMP]; return a.v > b.v; }
inline bool operator<=(cdouble a, cdouble b) { ++g_opcount[OC_CMP]; return a.v <= b.v; }
inline bool operator>=(cdouble a, cdouble b) { ++g_opcount[OC_CMP]; return a.v >= b.v; }
inline bool operator==(cdouble a, cdouble b) { ++g_opcount[OC_CMP]; return a.v == b.v; }
inline bool operator!=(cdouble a, cdouble b) { ++g_opcount[OC_CMP]; return a.v != b.v; }
inline cdouble sqrt(cdouble a) { ++g_opcount[OC_SQRT]; return cdouble(::sqrt(a.v)); }
inline cdouble exp(cdouble a) { ++g_opcount[OC_EXP]; return cdouble(::exp(a.v)); }
inline cdouble sin(cdouble a) { ++g_opcount[OC_TRIG]; return cdouble(::sin(a.v)); }
inline cdouble cos(cdouble a) { ++g_opcount[OC_TRIG]; return cdouble(::cos(a.v)); }
inline cdouble floor(cdouble a) { ++g_opcount[OC_MISC]; return cdouble(::floor(a.v)); }
inline cdouble fabs(cdouble a) { ++g_opcount[OC_MISC]; return cdouble(::fabs(a.v)); }
inline cdouble fmin(cdouble a, cdouble b) { ++g_opcount[OC_MISC]; return cdouble(::fmin(a.v, b.v)); }
inline cdouble nearbyint(cdouble a) { return cdouble(::nearbyint(a.v)); }      // diagnostics only
inline cdouble frexp(cdouble a, int *e) { return cdouble(::frexp(a.v, e)); }
inline cdouble ldexp(cdouble a, int e) { return cdouble(::ldexp(a.v, e)); }
inline bool oc_isfinite(cdouble a) { return ::isfinite(a.v); }
