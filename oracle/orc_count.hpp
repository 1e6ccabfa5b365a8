/*
 * orc_count.hpp — TEST INFRASTRUCTURE, part of the oracle.  An operation-counting stand-in for `double`.
 *
 * oracle/grpic_oracle.c is plain C.  Compiled a second time as C++ with -DORC_COUNT it sees
 * `#define double orc_cnt`: every +, -, *, /, comparison and math-library call of the statement of the method is then
 * executed on this class, which does the same FP64 arithmetic and counts it, per stage of the step (ORC_STAGE marks
 * in the source).  Nothing of the arithmetic changes; the count is of the oracle AS WRITTEN (no common
 * sub-expression is shared, the coordinate map and the metric are re-evaluated wherever the text evaluates them).
 * Used by oracle.count_ops() -> tests/test_oracle_opcount.py, bench.py's cpu_baseline leg, DESIGN.md section 7.
 */
#pragma once
#include <math.h>
#include <stdint.h>

enum { ORC_K_ADD = 0, ORC_K_MUL, ORC_K_DIV, ORC_K_SQRT, ORC_K_EXPLOG, ORC_K_SINCOS, ORC_K_FLOOR, ORC_K_MINMAX, ORC_K_CMP,
       ORC_K_NEG, ORC_N_KINDS };
enum { ORC_N_STAGES = 8 };

static thread_local int orc_stage_now = 0;
static thread_local int64_t orc_counts[ORC_N_STAGES][ORC_N_KINDS];
#define ORC_STAGE(s) (orc_stage_now = (s))
static inline void orc_tick(int kind) { ++orc_counts[orc_stage_now][kind]; }

struct orc_cnt {
  double v;
  orc_cnt() = default;
  orc_cnt(double x) : v(x) {}
  orc_cnt(int x) : v((double)x) {}
  orc_cnt(long x) : v((double)x) {}
  orc_cnt(long long x) : v((double)x) {}
  explicit operator int32_t() const { return (int32_t)v; }
  explicit operator int64_t() const { return (int64_t)v; }
  explicit operator bool() const { return v != 0.0; }
  orc_cnt& operator+=(const orc_cnt& o) { orc_tick(ORC_K_ADD); v += o.v; return *this; }
  orc_cnt& operator-=(const orc_cnt& o) { orc_tick(ORC_K_ADD); v -= o.v; return *this; }
  orc_cnt& operator*=(const orc_cnt& o) { orc_tick(ORC_K_MUL); v *= o.v; return *this; }
  orc_cnt& operator/=(const orc_cnt& o) { orc_tick(ORC_K_DIV); v /= o.v; return *this; }
};
static inline orc_cnt operator+(const orc_cnt& a, const orc_cnt& b) { orc_tick(ORC_K_ADD); return orc_cnt(a.v + b.v); }
static inline orc_cnt operator-(const orc_cnt& a, const orc_cnt& b) { orc_tick(ORC_K_ADD); return orc_cnt(a.v - b.v); }
static inline orc_cnt operator*(const orc_cnt& a, const orc_cnt& b) { orc_tick(ORC_K_MUL); return orc_cnt(a.v * b.v); }
static inline orc_cnt operator/(const orc_cnt& a, const orc_cnt& b) { orc_tick(ORC_K_DIV); return orc_cnt(a.v / b.v); }
static inline orc_cnt operator-(const orc_cnt& a) { orc_tick(ORC_K_NEG); return orc_cnt(-a.v); }
static inline bool operator<(const orc_cnt& a, const orc_cnt& b) { orc_tick(ORC_K_CMP); return a.v < b.v; }
static inline bool operator>(const orc_cnt& a, const orc_cnt& b) { orc_tick(ORC_K_CMP); return a.v > b.v; }
static inline bool operator<=(const orc_cnt& a, const orc_cnt& b) { orc_tick(ORC_K_CMP); return a.v <= b.v; }
static inline bool operator>=(const orc_cnt& a, const orc_cnt& b) { orc_tick(ORC_K_CMP); return a.v >= b.v; }
static inline bool operator==(const orc_cnt& a, const orc_cnt& b) { orc_tick(ORC_K_CMP); return a.v == b.v; }
static inline bool operator!=(const orc_cnt& a, const orc_cnt& b) { orc_tick(ORC_K_CMP); return a.v != b.v; }
static inline orc_cnt sqrt(const orc_cnt& a) { orc_tick(ORC_K_SQRT); return orc_cnt(::sqrt(a.v)); }
static inline orc_cnt exp(const orc_cnt& a) { orc_tick(ORC_K_EXPLOG); return orc_cnt(::exp(a.v)); }
static inline orc_cnt log(const orc_cnt& a) { orc_tick(ORC_K_EXPLOG); return orc_cnt(::log(a.v)); }
static inline orc_cnt sin(const orc_cnt& a) { orc_tick(ORC_K_SINCOS); return orc_cnt(::sin(a.v)); }
static inline orc_cnt cos(const orc_cnt& a) { orc_tick(ORC_K_SINCOS); return orc_cnt(::cos(a.v)); }
static inline orc_cnt tanh(const orc_cnt& a) { orc_tick(ORC_K_EXPLOG); return orc_cnt(::tanh(a.v)); }
static inline orc_cnt floor(const orc_cnt& a) { orc_tick(ORC_K_FLOOR); return orc_cnt(::floor(a.v)); }
static inline orc_cnt fabs(const orc_cnt& a) { orc_tick(ORC_K_NEG); return orc_cnt(::fabs(a.v)); }
static inline orc_cnt fmin(const orc_cnt& a, const orc_cnt& b) { orc_tick(ORC_K_MINMAX); return orc_cnt(::fmin(a.v, b.v)); }
static inline orc_cnt fmax(const orc_cnt& a, const orc_cnt& b) { orc_tick(ORC_K_MINMAX); return orc_cnt(::fmax(a.v, b.v)); }
static inline orc_cnt nextafter(const orc_cnt& a, const orc_cnt& b) { return orc_cnt(::nextafter(a.v, b.v)); }
