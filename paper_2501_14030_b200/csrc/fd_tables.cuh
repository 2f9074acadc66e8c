// fd_tables.cuh -- centred finite-difference weights as compile-time rationals (reading C11;
// PAPER.md:162 "rational constants ... moved to compile time", PAPER.md:168 orders 2-12).
// Unit grid spacing; the 1/dx and 1/dx^2 factors live in the coefficient planes.
//   first derivative :  sum_{k=1..NG} c1(k) (f[+k] - f[-k])
//   second derivative:  d2(0) f[0] + sum_{k=1..NG} d2(k) (f[+k] + f[-k])
// Standard tables (Fornberg, Math. Comp. 51 (1988) 699, Table 1), typed as literals here; with
// the loops over k fully unrolled the compiler folds every weight into an immediate.
#pragma once

#define HR_HD __host__ __device__ __forceinline__

template <int NG>
struct FdTable;

template <>
struct FdTable<1> {
  HR_HD static constexpr double c1(int k) {
    constexpr double t[2] = {0.0, 1.0 / 2.0};
    return t[k];
  }
  HR_HD static constexpr double d2(int k) {
    constexpr double t[2] = {-2.0, 1.0};
    return t[k];
  }
};

template <>
struct FdTable<2> {
  HR_HD static constexpr double c1(int k) {
    constexpr double t[3] = {0.0, 2.0 / 3.0, -1.0 / 12.0};
    return t[k];
  }
  HR_HD static constexpr double d2(int k) {
    constexpr double t[3] = {-5.0 / 2.0, 4.0 / 3.0, -1.0 / 12.0};
    return t[k];
  }
};

template <>
struct FdTable<3> {
  HR_HD static constexpr double c1(int k) {
    constexpr double t[4] = {0.0, 3.0 / 4.0, -3.0 / 20.0, 1.0 / 60.0};
    return t[k];
  }
  HR_HD static constexpr double d2(int k) {
    constexpr double t[4] = {-49.0 / 18.0, 3.0 / 2.0, -3.0 / 20.0, 1.0 / 90.0};
    return t[k];
  }
};

template <>
struct FdTable<4> {
  HR_HD static constexpr double c1(int k) {
    constexpr double t[5] = {0.0, 4.0 / 5.0, -1.0 / 5.0, 4.0 / 105.0, -1.0 / 280.0};
    return t[k];
  }
  HR_HD static constexpr double d2(int k) {
    constexpr double t[5] = {-205.0 / 72.0, 8.0 / 5.0, -1.0 / 5.0, 8.0 / 315.0, -1.0 / 560.0};
    return t[k];
  }
};

template <>
struct FdTable<5> {
  HR_HD static constexpr double c1(int k) {
    constexpr double t[6] = {0.0, 5.0 / 6.0, -5.0 / 21.0, 5.0 / 84.0, -5.0 / 504.0, 1.0 / 1260.0};
    return t[k];
  }
  HR_HD static constexpr double d2(int k) {
    constexpr double t[6] = {-5269.0 / 1800.0, 5.0 / 3.0, -5.0 / 21.0, 5.0 / 126.0, -5.0 / 1008.0, 1.0 / 3150.0};
    return t[k];
  }
};

template <>
struct FdTable<6> {
  HR_HD static constexpr double c1(int k) {
    constexpr double t[7] = {0.0, 6.0 / 7.0, -15.0 / 56.0, 5.0 / 63.0, -1.0 / 56.0, 1.0 / 385.0, -1.0 / 5544.0};
    return t[k];
  }
  HR_HD static constexpr double d2(int k) {
    constexpr double t[7] = {-5369.0 / 1800.0, 12.0 / 7.0, -15.0 / 56.0, 10.0 / 189.0, -1.0 / 112.0, 2.0 / 1925.0, -1.0 / 16632.0};
    return t[k];
  }
};
