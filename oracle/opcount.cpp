// oracle/opcount.cpp -- TEST / MEASUREMENT INFRASTRUCTURE, NOT PRODUCT CODE.
// Instantiates the oracle (lbr_oracle.hpp) on an op-counting scalar type to obtain the ALGORITHMIC fp64 work per row
// ("+ - x" = 1 flop each, "/" and sqrt = 1 each and reported separately, calls to
// exp/log/log1p/erfc/erfcx/Phi^-1/cbrt counted as calls).  bench.py / DESIGN.md convert calls to flops with a per-call
// cost table.  Counting uses fixed_iters = 2 (the GPU's Householder count).
#include <cstdint>
#include <cstring>

#include "lbr_oracle.hpp"

namespace lbr_oracle {

enum { C_ADD, C_MUL, C_DIV, C_SQRT, C_EXP, C_LOG, C_LOG1P, C_ERFC, C_ERFCX, C_NINV, C_CBRT, C_N };
static thread_local uint64_t g_cnt[C_N];

struct Cnt {
  double v;
  Cnt() : v(0) {}
  Cnt(double d) : v(d) {}
  Cnt(long double d) : v((double)d) {}
  Cnt(int d) : v(d) {}
  explicit operator double() const { return v; }
  explicit operator long double() const { return v; }
};
inline Cnt operator+(Cnt a, Cnt b) { ++g_cnt[C_ADD]; return Cnt(a.v + b.v); }
inline Cnt operator-(Cnt a, Cnt b) { ++g_cnt[C_ADD]; return Cnt(a.v - b.v); }
inline Cnt operator*(Cnt a, Cnt b) { ++g_cnt[C_MUL]; return Cnt(a.v * b.v); }
inline Cnt operator/(Cnt a, Cnt b) { ++g_cnt[C_DIV]; return Cnt(a.v / b.v); }
inline Cnt operator-(Cnt a) { return Cnt(-a.v); }
inline Cnt& operator+=(Cnt& a, Cnt b) { a = a + b; return a; }
inline Cnt& operator-=(Cnt& a, Cnt b) { a = a - b; return a; }
inline Cnt& operator*=(Cnt& a, Cnt b) { a = a * b; return a; }
inline bool operator<(Cnt a, Cnt b) { return a.v < b.v; }
inline bool operator>(Cnt a, Cnt b) { return a.v > b.v; }
inline bool operator<=(Cnt a, Cnt b) { return a.v <= b.v; }
inline bool operator>=(Cnt a, Cnt b) { return a.v >= b.v; }
inline bool operator==(Cnt a, Cnt b) { return a.v == b.v; }
inline bool operator!=(Cnt a, Cnt b) { return a.v != b.v; }
inline Cnt exp(Cnt a) { ++g_cnt[C_EXP]; return Cnt(std::exp(a.v)); }
inline Cnt log(Cnt a) { ++g_cnt[C_LOG]; return Cnt(std::log(a.v)); }
inline Cnt log1p(Cnt a) { ++g_cnt[C_LOG1P]; return Cnt(std::log1p(a.v)); }
inline Cnt sqrt(Cnt a) { ++g_cnt[C_SQRT]; return Cnt(std::sqrt(a.v)); }
inline Cnt erfc(Cnt a) { ++g_cnt[C_ERFC]; return Cnt(std::erfc(a.v)); }
inline Cnt cbrt(Cnt a) { ++g_cnt[C_CBRT]; return Cnt(std::cbrt(a.v)); }
inline Cnt fabs(Cnt a) { return Cnt(std::fabs(a.v)); }
inline Cnt acos(Cnt a) { return Cnt(std::acos(a.v)); }   // only used to spell pi: a constant, not counted
inline bool isfinite(Cnt a) { return std::isfinite(a.v); }
template <> inline Cnt erfcx_<Cnt>(Cnt z) { ++g_cnt[C_ERFCX]; return Cnt((double)erfcx_ld((long double)z.v)); }
template <> inline Cnt ninv_<Cnt>(Cnt p) { ++g_cnt[C_NINV]; return Cnt((double)ninv_ld((long double)p.v)); }
// constants are compile-time values on any real implementation: do not count the ops that spell them
template <> struct K<Cnt> {
  static Cnt pi() { return Cnt(K<double>::pi()); }
  static Cnt sqrt2() { return Cnt(K<double>::sqrt2()); }
  static Cnt sqrt3() { return Cnt(K<double>::sqrt3()); }
  static Cnt phi0() { return Cnt(K<double>::phi0()); }
  static Cnt sqrt_pi_2() { return Cnt(K<double>::sqrt_pi_2()); }
};
template <> inline Cnt ln_v<Cnt>(Cnt h, Cnt t) { return Cnt(std::log(K<double>::phi0())) - Cnt(0.5) * (h * h + t * t); }

}  // namespace lbr_oracle

namespace std {
template <> struct numeric_limits<lbr_oracle::Cnt> {
  static lbr_oracle::Cnt quiet_NaN() { return lbr_oracle::Cnt(numeric_limits<double>::quiet_NaN()); }
  static lbr_oracle::Cnt infinity() { return lbr_oracle::Cnt(numeric_limits<double>::infinity()); }
  static lbr_oracle::Cnt epsilon() { return lbr_oracle::Cnt(numeric_limits<double>::epsilon()); }
};
}  // namespace std

using namespace lbr_oracle;

extern "C" {
// counts[5][C_N]: per class c = zone 0..3 of OK rows, c = 4 all non-OK rows;  rows[5]: rows per class.
void oracle_count_ops(int64_t n, const double* SorF, const double* Kk, const double* tau, const double* r,
                      const double* q, const double* P, const double* flag, int fixed_iters, uint64_t* counts,
                      uint64_t* rows) {
  std::memset(counts, 0, sizeof(uint64_t) * 5 * C_N);
  std::memset(rows, 0, sizeof(uint64_t) * 5);
  for (int64_t i = 0; i < n; ++i) {
    std::memset(g_cnt, 0, sizeof(g_cnt));
    Cnt rr = r ? Cnt(r[i]) : Cnt(0.0), qq = q ? Cnt(q[i]) : Cnt(0.0);
    RowResult<Cnt> o = lbr_row<Cnt>(Cnt(SorF[i]), Cnt(Kk[i]), Cnt(tau[i]), (r && q) ? &rr : nullptr,
                                    (r && q) ? &qq : nullptr, Cnt(P[i]), Cnt(flag[i]), fixed_iters);
    const int c = (o.status == ST_OK) ? o.zone : 4;
    for (int k = 0; k < C_N; ++k) counts[c * C_N + k] += g_cnt[k];
    ++rows[c];
  }
}
int oracle_count_ops_ncounters(void) { return C_N; }
}
