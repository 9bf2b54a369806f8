// fft_codelets.cuh -- fully unrolled in-register FFTs of length 16 / 24 / 32 / 48.
//
// Plain Cooley-Tukey, N = N1 * N2 (input index N2 n1 + n2, output index k1 + N1 k2):
//   X[k1 + N1 k2] = sum_{n2} W_N^{n2 k1} ( sum_{n1} x[N2 n1 + n2] W_N1^{n1 k1} ) W_N2^{n2 k2}
// with radix 2 / 3 / 4 butterflies at the leaves.  Every index and every twiddle is a compile
// time constant (static_for over integral_constant, constexpr cos/sin), so the arrays live in
// registers and twiddles become FFMA immediates.  W_N = exp(-2 pi i / N) forward, conjugate
// when INV.  Natural order in, natural order out, no scaling.
#pragma once
#include <cuda_runtime.h>

#include <type_traits>
#include <utility>

namespace idg {
namespace fft {

template <int I, int END, class F>
__device__ __forceinline__ void static_for(F &&f) {
  if constexpr (I < END) {
    f(std::integral_constant<int, I>{});
    static_for<I + 1, END>(f);
  }
}

// constexpr cos / sin of 2 pi j / n by Taylor series in double (argument reduced to (-pi, pi])
constexpr double kPi = 3.14159265358979323846264338327950288;
__host__ __device__ constexpr double reduced_angle(int j, int n) {
  int r = ((j % n) + n) % n;
  if (2 * r > n) r -= n;
  return 2.0 * kPi * (double)r / (double)n;
}
__host__ __device__ constexpr double taylor_cos(double a) {
  double term = 1.0, sum = 1.0;
  for (int k = 1; k < 20; ++k) {
    term *= -a * a / (double)((2 * k - 1) * (2 * k));
    sum += term;
  }
  return sum;
}
__host__ __device__ constexpr double taylor_sin(double a) {
  double term = a, sum = a;
  for (int k = 1; k < 20; ++k) {
    term *= -a * a / (double)((2 * k) * (2 * k + 1));
    sum += term;
  }
  return sum;
}
// exact values on the axes and diagonals keep the butterflies free of round-off dust
__host__ __device__ constexpr double tw_cos(int j, int n) {
  const int r = ((j % n) + n) % n;
  if (4 * r == n || 4 * r == 3 * n) return 0.0;
  if (r == 0) return 1.0;
  if (2 * r == n) return -1.0;
  return taylor_cos(reduced_angle(j, n));
}
__host__ __device__ constexpr double tw_sin(int j, int n) {
  const int r = ((j % n) + n) % n;
  if (r == 0 || 2 * r == n) return 0.0;
  if (4 * r == n) return 1.0;
  if (4 * r == 3 * n) return -1.0;
  return taylor_sin(reduced_angle(j, n));
}

// x * W_N^J
template <int J, int N, bool INV>
__device__ __forceinline__ float2 twiddle(float2 x) {
  constexpr int r = ((J % N) + N) % N;
  if constexpr (r == 0) {
    return x;
  } else if constexpr (2 * r == N) {
    return make_float2(-x.x, -x.y);
  } else if constexpr (4 * r == N) {  // forward: -i ; inverse: +i
    return INV ? make_float2(-x.y, x.x) : make_float2(x.y, -x.x);
  } else if constexpr (4 * r == 3 * N) {
    return INV ? make_float2(x.y, -x.x) : make_float2(-x.y, x.x);
  } else {
    constexpr float c = (float)tw_cos(r, N);
    constexpr float s = (float)(INV ? tw_sin(r, N) : -tw_sin(r, N));
    return make_float2(x.x * c - x.y * s, x.x * s + x.y * c);
  }
}

template <int N, bool INV>
struct Fft;

template <bool INV>
struct Fft<2, INV> {
  static __device__ __forceinline__ void run(float2 (&x)[2]) {
    const float2 a = x[0], b = x[1];
    x[0] = make_float2(a.x + b.x, a.y + b.y);
    x[1] = make_float2(a.x - b.x, a.y - b.y);
  }
};

template <bool INV>
struct Fft<3, INV> {
  static __device__ __forceinline__ void run(float2 (&x)[3]) {
    constexpr float h = 0.86602540378443864676f;  // sin(pi/3)
    const float2 a = x[0], b = x[1], c = x[2];
    const float2 s = make_float2(b.x + c.x, b.y + c.y), d = make_float2(b.x - c.x, b.y - c.y);
    const float2 m = make_float2(a.x - 0.5f * s.x, a.y - 0.5f * s.y);
    // forward: X1 = m - i h d, X2 = m + i h d ; inverse swaps
    const float2 r = make_float2(h * d.y, -h * d.x);  // -i h d
    x[0] = make_float2(a.x + s.x, a.y + s.y);
    if (INV) {
      x[1] = make_float2(m.x - r.x, m.y - r.y);
      x[2] = make_float2(m.x + r.x, m.y + r.y);
    } else {
      x[1] = make_float2(m.x + r.x, m.y + r.y);
      x[2] = make_float2(m.x - r.x, m.y - r.y);
    }
  }
};

template <bool INV>
struct Fft<4, INV> {
  static __device__ __forceinline__ void run(float2 (&x)[4]) {
    const float2 a = x[0], b = x[1], c = x[2], d = x[3];
    const float2 s0 = make_float2(a.x + c.x, a.y + c.y), d0 = make_float2(a.x - c.x, a.y - c.y);
    const float2 s1 = make_float2(b.x + d.x, b.y + d.y), d1 = make_float2(b.x - d.x, b.y - d.y);
    // -i d1 forward, +i d1 inverse
    const float2 r = INV ? make_float2(-d1.y, d1.x) : make_float2(d1.y, -d1.x);
    x[0] = make_float2(s0.x + s1.x, s0.y + s1.y);
    x[1] = make_float2(d0.x + r.x, d0.y + r.y);
    x[2] = make_float2(s0.x - s1.x, s0.y - s1.y);
    x[3] = make_float2(d0.x - r.x, d0.y - r.y);
  }
};

template <int N1, int N2, bool INV>
__device__ __forceinline__ void cooley_tukey(float2 (&x)[N1 * N2]) {
  constexpr int N = N1 * N2;
  float2 y[N];
  static_for<0, N2>([&](auto n2c) {
    constexpr int n2 = decltype(n2c)::value;
    float2 t[N1];
    static_for<0, N1>([&](auto n1c) { constexpr int n1 = decltype(n1c)::value; t[n1] = x[N2 * n1 + n2]; });
    Fft<N1, INV>::run(t);
    static_for<0, N1>([&](auto k1c) {
      constexpr int k1 = decltype(k1c)::value;
      y[k1 * N2 + n2] = twiddle<n2 * k1, N, INV>(t[k1]);
    });
  });
  static_for<0, N1>([&](auto k1c) {
    constexpr int k1 = decltype(k1c)::value;
    float2 s[N2];
    static_for<0, N2>([&](auto n2c) { constexpr int n2 = decltype(n2c)::value; s[n2] = y[k1 * N2 + n2]; });
    Fft<N2, INV>::run(s);
    static_for<0, N2>([&](auto k2c) { constexpr int k2 = decltype(k2c)::value; x[k1 + N1 * k2] = s[k2]; });
  });
}

template <bool INV> struct Fft<8, INV>  { static __device__ __forceinline__ void run(float2 (&x)[8])  { cooley_tukey<2, 4, INV>(x); } };
template <bool INV> struct Fft<16, INV> { static __device__ __forceinline__ void run(float2 (&x)[16]) { cooley_tukey<4, 4, INV>(x); } };
template <bool INV> struct Fft<24, INV> { static __device__ __forceinline__ void run(float2 (&x)[24]) { cooley_tukey<3, 8, INV>(x); } };
template <bool INV> struct Fft<32, INV> { static __device__ __forceinline__ void run(float2 (&x)[32]) { cooley_tukey<4, 8, INV>(x); } };
template <bool INV> struct Fft<48, INV> { static __device__ __forceinline__ void run(float2 (&x)[48]) { cooley_tukey<3, 16, INV>(x); } };

}  // namespace fft
}  // namespace idg
