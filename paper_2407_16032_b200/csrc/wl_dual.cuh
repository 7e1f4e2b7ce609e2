// wl_dual.cuh -- scalar types of the generic engine (wl_generic.cu): double, and a forward-mode dual number that carries
// one derivative lane d/d(theta) beside the value ("automatic differentiation", "running the code with a
// T = Dual data-type holding the value and derivative simultaneously ... the exact derivative (not a finite-difference
// approximation)").  Comparisons and branches look at the value only, so the derivative follows the branch the value takes.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

struct Dual {
    double v, d;
    __host__ __device__ Dual() : v(0.0), d(0.0) {}
    __host__ __device__ Dual(double v_) : v(v_), d(0.0) {}
    __host__ __device__ Dual(double v_, double d_) : v(v_), d(d_) {}
};

__host__ __device__ inline Dual operator+(const Dual& a, const Dual& b) { return Dual(a.v + b.v, a.d + b.d); }
__host__ __device__ inline Dual operator-(const Dual& a, const Dual& b) { return Dual(a.v - b.v, a.d - b.d); }
__host__ __device__ inline Dual operator-(const Dual& a) { return Dual(-a.v, -a.d); }
__host__ __device__ inline Dual operator*(const Dual& a, const Dual& b) { return Dual(a.v * b.v, a.d * b.v + a.v * b.d); }
__host__ __device__ inline Dual operator/(const Dual& a, const Dual& b)
{
    const double q = a.v / b.v;
    return Dual(q, (a.d - q * b.d) / b.v);
}
__host__ __device__ inline Dual& operator+=(Dual& a, const Dual& b) { a.v += b.v; a.d += b.d; return a; }
__host__ __device__ inline Dual& operator-=(Dual& a, const Dual& b) { a.v -= b.v; a.d -= b.d; return a; }
__host__ __device__ inline bool operator<(const Dual& a, const Dual& b) { return a.v < b.v; }
__host__ __device__ inline bool operator>(const Dual& a, const Dual& b) { return a.v > b.v; }
__host__ __device__ inline bool operator<=(const Dual& a, const Dual& b) { return a.v <= b.v; }
__host__ __device__ inline bool operator>=(const Dual& a, const Dual& b) { return a.v >= b.v; }

// elementary functions for both scalar types
__host__ __device__ inline double g_sqrt(double a) { return sqrt(a); }
__host__ __device__ inline double g_sin(double a) { return sin(a); }
__host__ __device__ inline double g_cos(double a) { return cos(a); }
__host__ __device__ inline double g_abs(double a) { return fabs(a); }
__host__ __device__ inline double g_val(double a) { return a; }
__host__ __device__ inline double g_der(double) { return 0.0; }
__host__ __device__ inline Dual g_sqrt(const Dual& a) { const double s = sqrt(a.v); return Dual(s, s > 0.0 ? 0.5 * a.d / s : 0.0); }
__host__ __device__ inline Dual g_sin(const Dual& a) { return Dual(sin(a.v), cos(a.v) * a.d); }
__host__ __device__ inline Dual g_cos(const Dual& a) { return Dual(cos(a.v), -sin(a.v) * a.d); }
__host__ __device__ inline Dual g_abs(const Dual& a) { return a.v < 0.0 ? -a : a; }
__host__ __device__ inline double g_val(const Dual& a) { return a.v; }
__host__ __device__ inline double g_der(const Dual& a) { return a.d; }

template <class T> struct Lanes;                 // how many doubles a scalar is made of (reductions work lane by lane)
template <> struct Lanes<double> {
    static const int N = 1;
    __host__ __device__ static double get(const double& a, int) { return a; }
    __host__ __device__ static double make(const double* l) { return l[0]; }
};
template <> struct Lanes<Dual> {
    static const int N = 2;
    __host__ __device__ static double get(const Dual& a, int k) { return k == 0 ? a.v : a.d; }
    __host__ __device__ static Dual make(const double* l) { return Dual(l[0], l[1]); }
};
