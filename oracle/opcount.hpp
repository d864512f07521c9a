// op-counting scalar for the oracle (audit of the fp64 operation mix per layer.point; not part of the oracle proper)
#pragma once
#include <cmath>
#include <type_traits>
struct OpCounts { long long add, mul, div, sqrt_, exp_, log_, cmp; };
extern thread_local OpCounts g_ops;
struct Counted {
  long double v;
  Counted() = default;
  template <class T, class = typename std::enable_if<std::is_arithmetic<T>::value>::type> Counted(T x) : v((long double)x) {}
  explicit operator double() const { return (double)v; }
  explicit operator long double() const { return v; }
  explicit operator int() const { return (int)v; }
  explicit operator bool() const { return v != 0; }
};
#define OPC_BIN(op, field) \
  inline Counted operator op(Counted a, Counted b) { ++g_ops.field; Counted r; r.v = a.v op b.v; return r; } \
  template <class T, class = typename std::enable_if<std::is_arithmetic<T>::value>::type> inline Counted operator op(Counted a, T b) { return a op Counted(b); } \
  template <class T, class = typename std::enable_if<std::is_arithmetic<T>::value>::type> inline Counted operator op(T a, Counted b) { return Counted(a) op b; }
OPC_BIN(+, add) OPC_BIN(-, add) OPC_BIN(*, mul) OPC_BIN(/, div)
inline Counted operator-(Counted a) { Counted r; r.v = -a.v; return r; }
inline Counted operator+(Counted a) { return a; }
inline Counted &operator+=(Counted &a, Counted b) { a = a + b; return a; }
inline Counted &operator-=(Counted &a, Counted b) { a = a - b; return a; }
inline Counted &operator*=(Counted &a, Counted b) { a = a * b; return a; }
inline Counted &operator/=(Counted &a, Counted b) { a = a / b; return a; }
#define OPC_CMP(op) \
  inline bool operator op(Counted a, Counted b) { ++g_ops.cmp; return a.v op b.v; } \
  template <class T, class = typename std::enable_if<std::is_arithmetic<T>::value>::type> inline bool operator op(Counted a, T b) { ++g_ops.cmp; return a.v op (long double)b; } \
  template <class T, class = typename std::enable_if<std::is_arithmetic<T>::value>::type> inline bool operator op(T a, Counted b) { ++g_ops.cmp; return (long double)a op b.v; }
OPC_CMP(<) OPC_CMP(>) OPC_CMP(<=) OPC_CMP(>=) OPC_CMP(==) OPC_CMP(!=)
inline bool operator!(Counted a) { return a.v == 0; }
inline Counted exp(Counted a) { ++g_ops.exp_; Counted r; r.v = expl(a.v); return r; }
inline Counted sqrt(Counted a) { ++g_ops.sqrt_; Counted r; r.v = sqrtl(a.v); return r; }
inline Counted log(Counted a) { ++g_ops.log_; Counted r; r.v = logl(a.v); return r; }
inline Counted log10(Counted a) { ++g_ops.log_; Counted r; r.v = log10l(a.v); return r; }
inline Counted fabs(Counted a) { Counted r; r.v = fabsl(a.v); return r; }
