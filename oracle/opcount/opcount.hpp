// opcount.hpp -- an operation-counting stand-in for `double`, used to count the ALGORITHMIC
// floating-point operations of the oracle's own arithmetic (test / measurement infrastructure,
// see oracle/mmo.h).  Each + - * / sqrt exp pow counts 1; comparisons, fabs,
// negation, min/max selections and copies count 0.  Same size and layout as double.
#pragma once
#include <cmath>

struct cnt {
    double v;
    static long long ops;
    cnt() = default;
    cnt(double x) : v(x) {}
    cnt(int x) : v(x) {}
    cnt(long long x) : v((double)x) {}
    cnt(unsigned long x) : v((double)x) {}
};
inline long long cnt::ops = 0;
static_assert(sizeof(cnt) == sizeof(double), "cnt must mirror double");

#define MMO_BINOP(op)                                                                  \
    inline cnt operator op(cnt a, cnt b) { ++cnt::ops; return cnt(a.v op b.v); }       \
    inline cnt operator op(cnt a, double b) { ++cnt::ops; return cnt(a.v op b); }      \
    inline cnt operator op(double a, cnt b) { ++cnt::ops; return cnt(a op b.v); }      \
    inline cnt operator op(cnt a, int b) { ++cnt::ops; return cnt(a.v op b); }         \
    inline cnt operator op(int a, cnt b) { ++cnt::ops; return cnt(a op b.v); }
MMO_BINOP(+) MMO_BINOP(-) MMO_BINOP(*) MMO_BINOP(/)
#undef MMO_BINOP
inline cnt operator-(cnt a) { return cnt(-a.v); }
inline cnt& operator+=(cnt& a, cnt b) { ++cnt::ops; a.v += b.v; return a; }
inline cnt& operator-=(cnt& a, cnt b) { ++cnt::ops; a.v -= b.v; return a; }
inline cnt& operator*=(cnt& a, cnt b) { ++cnt::ops; a.v *= b.v; return a; }
inline cnt& operator/=(cnt& a, cnt b) { ++cnt::ops; a.v /= b.v; return a; }
#define MMO_CMP(op)                                                    \
    inline bool operator op(cnt a, cnt b) { return a.v op b.v; }       \
    inline bool operator op(cnt a, double b) { return a.v op b; }      \
    inline bool operator op(double a, cnt b) { return a op b.v; }
MMO_CMP(<) MMO_CMP(>) MMO_CMP(<=) MMO_CMP(>=) MMO_CMP(==) MMO_CMP(!=)
#undef MMO_CMP
inline bool operator!(cnt a) { return !a.v; }
inline cnt sqrt(cnt a) { ++cnt::ops; return cnt(std::sqrt(a.v)); }
inline cnt exp(cnt a) { ++cnt::ops; return cnt(std::exp(a.v)); }
inline cnt pow(cnt a, double b) { ++cnt::ops; return cnt(std::pow(a.v, b)); }
inline cnt pow(cnt a, cnt b) { ++cnt::ops; return cnt(std::pow(a.v, b.v)); }
inline cnt fabs(cnt a) { return cnt(std::fabs(a.v)); }
inline bool mmo_isfinite(cnt a) { return std::isfinite(a.v); }
