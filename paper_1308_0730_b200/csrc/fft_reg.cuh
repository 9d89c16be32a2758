// Register-resident mixed-radix FFTs of compile-time length (2..36, 2-3-5-7-smooth).
//
// Every pencil transform of the multi-view Richardson-Lucy path (the
// integrals of eq. 1/2 are convolutions, evaluated through the convolution theorem) is a
// length-M = A*B DFT split into an A-point and a B-point transform that each live in the
// registers of one thread; only the A<->B transposition goes through shared memory.
// This header is those A- and B-point transforms.  All indices and twiddle factors are
// compile-time constants (static_for + constexpr trigonometry evaluated in double), so the
// generated code is straight-line FADD/FMUL/FFMA with immediate operands.
//
// The file is plain C++17 when MVD_HOST_TEST is defined (the butterflies can then be
// checked on the CPU against a DFT); under nvcc everything is __device__ __forceinline__.
#pragma once

#include <type_traits>

#ifdef MVD_HOST_TEST
#include <cmath>
struct float2 { float x, y; };
static inline float2 make_float2(float a, float b) { return float2{a, b}; }
#define MVD_DEV inline
#define MVD_CE constexpr
#define MVD_FMA(a, b, c) std::fmaf((a), (b), (c))
#define MVD_MUL(a, b) ((a) * (b))
#else
#include <cuda_runtime.h>
#define MVD_DEV __device__ __forceinline__
#define MVD_CE __host__ __device__ constexpr
// explicit rounding: the complex products contract the same way in every kernel, so the same
// transform gives bit-identical results wherever it is inlined (resume == uninterrupted run)
#define MVD_FMA(a, b, c) __fmaf_rn((a), (b), (c))
#define MVD_MUL(a, b) __fmul_rn((a), (b))
#endif

namespace mvd {

// ---------------------------------------------------------------------------------------
// compile-time loop
// ---------------------------------------------------------------------------------------
template <int I, int N, class F>
MVD_DEV void static_for(F&& f) {
  if constexpr (I < N) {
    f(std::integral_constant<int, I>{});
    static_for<I + 1, N>(f);
  }
}

// ---------------------------------------------------------------------------------------
// constexpr roots of unity: exp(2*pi*i*k/n), evaluated in double, exact at multiples of 1/8 turn
// ---------------------------------------------------------------------------------------
struct cdouble { double re, im; };

constexpr double kPi = 3.141592653589793238462643383279502884;

MVD_CE double ce_sin_small(double x) {   // |x| <= pi/4, Taylor to x^27
  double x2 = x * x, term = x, sum = x;
  for (int i = 1; i <= 13; ++i) { term *= -x2 / double((2 * i) * (2 * i + 1)); sum += term; }
  return sum;
}
MVD_CE double ce_cos_small(double x) {   // |x| <= pi/4, Taylor to x^26
  double x2 = x * x, term = 1.0, sum = 1.0;
  for (int i = 1; i <= 13; ++i) { term *= -x2 / double((2 * i - 1) * (2 * i)); sum += term; }
  return sum;
}
MVD_CE cdouble ce_root(long long k, long long n) {   // exp(+2*pi*i*k/n)
  k %= n;
  if (k < 0) k += n;
  // nearest quarter turn q, remainder angle pi*(4k - q n)/(2n) in [-pi/4, pi/4]
  long long q = (8 * k + n) / (2 * n);
  long long rnum = 4 * k - q * n;
  double c = 1.0, s = 0.0;
  if (rnum != 0) {
    if (2 * rnum == n)       { c = 0.70710678118654752440; s = 0.70710678118654752440; }
    else if (2 * rnum == -n) { c = 0.70710678118654752440; s = -0.70710678118654752440; }
    else { double th = kPi * double(rnum) / double(2 * n); c = ce_cos_small(th); s = ce_sin_small(th); }
  }
  switch (q & 3) {
    case 0: return cdouble{c, s};
    case 1: return cdouble{-s, c};
    case 2: return cdouble{-c, -s};
    default: return cdouble{s, -c};
  }
}

// ---------------------------------------------------------------------------------------
// complex helpers
// ---------------------------------------------------------------------------------------
#if defined(MVD_HOST_TEST) || defined(MVD_NO_F32X2)
MVD_DEV float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
MVD_DEV float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
// a + c * s, c real
MVD_DEV float2 caxpy(float c, float2 s, float2 a) { return make_float2(MVD_FMA(c, s.x, a.x), MVD_FMA(c, s.y, a.y)); }
MVD_DEV float2 cscale(float c, float2 s) { return make_float2(c * s.x, c * s.y); }
MVD_DEV float2 fma2(float ax, float ay, float bx, float by, float cx, float cy) {
  return make_float2(MVD_FMA(ax, bx, cx), MVD_FMA(ay, by, cy));
}
MVD_DEV float2 mul2(float ax, float ay, float bx, float by) { return make_float2(MVD_MUL(ax, bx), MVD_MUL(ay, by)); }
#else
// sm_100a packed fp32: one FADD2 / FFMA2 / FMUL2 handles the real and the imaginary part together
// (IEEE per lane, so results equal the scalar forms bit for bit); halves the issue slots of the
// butterflies, which is what the x pass is short of.
// (ax,ay) * (bx,by) + (cx,cy) and (ax,ay) * (bx,by): the operands may repeat or swap the halves of a
// register pair (SASS operand modes .F32 broadcast, .F32x2.LO_HI swap), so neither costs a move
MVD_DEV float2 fma2(float ax, float ay, float bx, float by, float cx, float cy) {
  float2 r;
  asm("{.reg .b64 ra, rb, rc, rd; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; mov.b64 rc, {%6,%7}; fma.rn.f32x2 rd, ra, rb, rc; mov.b64 {%0,%1}, rd;}"
      : "=f"(r.x), "=f"(r.y) : "f"(ax), "f"(ay), "f"(bx), "f"(by), "f"(cx), "f"(cy));
  return r;
}
MVD_DEV float2 mul2(float ax, float ay, float bx, float by) {
  float2 r;
  asm("{.reg .b64 ra, rb, rd; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; mul.rn.f32x2 rd, ra, rb; mov.b64 {%0,%1}, rd;}"
      : "=f"(r.x), "=f"(r.y) : "f"(ax), "f"(ay), "f"(bx), "f"(by));
  return r;
}
MVD_DEV float2 cadd(float2 a, float2 b) {
  float2 r;
  asm("{.reg .b64 ra, rb, rc; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; add.rn.f32x2 rc, ra, rb; mov.b64 {%0,%1}, rc;}"
      : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
  return r;
}
MVD_DEV float2 csub(float2 a, float2 b) {
  float2 r;
  asm("{.reg .b64 ra, rb, rc; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; sub.rn.f32x2 rc, ra, rb; mov.b64 {%0,%1}, rc;}"
      : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
  return r;
}
MVD_DEV float2 caxpy(float c, float2 s, float2 a) {   // a + c * s, c real
  float2 r;
  asm("{.reg .b64 rs, rc, ra, rd; mov.b64 rs, {%2,%3}; mov.b64 rc, {%4,%4}; mov.b64 ra, {%5,%6}; fma.rn.f32x2 rd, rs, rc, ra; mov.b64 {%0,%1}, rd;}"
      : "=f"(r.x), "=f"(r.y) : "f"(s.x), "f"(s.y), "f"(c), "f"(a.x), "f"(a.y));
  return r;
}
MVD_DEV float2 cscale(float c, float2 s) {
  float2 r;
  asm("{.reg .b64 rs, rc, rd; mov.b64 rs, {%2,%3}; mov.b64 rc, {%4,%4}; mul.rn.f32x2 rd, rs, rc; mov.b64 {%0,%1}, rd;}"
      : "=f"(r.x), "=f"(r.y) : "f"(s.x), "f"(s.y), "f"(c));
  return r;
}
#endif
// a * b and a * conj(b): one packed multiply a.x * (b.x, b.y) and two scalar FMAs for the a.y terms
// (no sign flip, no constant pair to build); the order of operations is fixed, so every kernel
// rounds a product the same way
MVD_DEV float2 cmul(float2 a, float2 b) {
  const float2 t = mul2(a.x, a.x, b.x, b.y);
  return make_float2(MVD_FMA(-a.y, b.y, t.x), MVD_FMA(a.y, b.x, t.y));
}
MVD_DEV float2 cmul_conj(float2 a, float2 b) {   // a * conj(b) = (a.x b.x + a.y b.y, a.y b.x - a.x b.y)
  const float2 t = mul2(a.y, a.y, b.y, b.x);
  return make_float2(MVD_FMA(a.x, b.x, t.x), MVD_FMA(-a.x, b.y, t.y));
}
// multiply by exp(DIR * 2*pi*i * K / N), K and N compile-time (DIR = -1 forward, +1 inverse)
template <int K, int N, int DIR>
MVD_DEV float2 cmul_root(float2 a) {
  constexpr int k = ((K % N) + N) % N;
  if constexpr (k == 0) {
    return a;
  } else if constexpr (4 * k == N) {          // * (DIR * i)
    return DIR > 0 ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
  } else if constexpr (2 * k == N) {          // * -1
    return make_float2(-a.x, -a.y);
  } else if constexpr (4 * k == 3 * N) {      // * (-DIR * i)
    return DIR > 0 ? make_float2(a.y, -a.x) : make_float2(-a.y, a.x);
  } else {
    constexpr cdouble w = ce_root(k, N);
    constexpr float c = float(w.re);
    constexpr float s = float(DIR > 0 ? w.im : -w.im);
    const float2 t = mul2(a.x, a.y, c, c);            // packed multiply by the broadcast immediate c
    return make_float2(MVD_FMA(-s, a.y, t.x), MVD_FMA(s, a.x, t.y));
  }
}

// ---------------------------------------------------------------------------------------
// prime-radix butterflies, in place, natural order
// ---------------------------------------------------------------------------------------
template <int DIR>
MVD_DEV void bfly2(float2& a, float2& b) {
  float2 t = csub(a, b);
  a = cadd(a, b);
  b = t;
}

template <int DIR>
MVD_DEV void bfly4(float2& a, float2& b, float2& c, float2& d) {
  float2 s0 = cadd(a, c), d0 = csub(a, c);
  float2 s1 = cadd(b, d), d1 = csub(b, d);
  a = cadd(s0, s1);
  c = csub(s0, s1);
  // b = d0 + DIR*i*d1, d = d0 - DIR*i*d1 with i*d1 = (-d1.y, d1.x)
  // b = d0 + DIR*i*d1, d = d0 - DIR*i*d1 with i*d1 = (-d1.y, d1.x): swapped operand, sign pair constant
  constexpr float sg = DIR > 0 ? 1.f : -1.f;
  b = fma2(d1.y, d1.x, -sg, sg, d0.x, d0.y);
  d = fma2(d1.y, d1.x, sg, -sg, d0.x, d0.y);
}

// odd prime P: pairs (m, P-m).  X_j = a_j + i*DIR*b_j, X_{P-j} = a_j - i*DIR*b_j with
// a_j = x0 + sum_m cos(2 pi j m/P) (x_m + x_{P-m}),  b_j = sum_m sin(2 pi j m/P) (x_m - x_{P-m}).
template <int P, int DIR>
MVD_DEV void bfly_odd(float2 (&x)[P]) {
  constexpr int H = (P - 1) / 2;
  float2 s[H], d[H];
  static_for<0, H>([&](auto m_) {
    constexpr int m = decltype(m_)::value + 1;
    s[m - 1] = cadd(x[m], x[P - m]);
    d[m - 1] = csub(x[m], x[P - m]);
  });
  float2 x0 = x[0];
  float2 sum = x0;
  static_for<0, H>([&](auto m_) { sum = cadd(sum, s[decltype(m_)::value]); });
  x[0] = sum;
  static_for<0, H>([&](auto j_) {
    constexpr int j = decltype(j_)::value + 1;
    float2 a = x0, b = make_float2(0.f, 0.f);
    static_for<0, H>([&](auto m_) {
      constexpr int m = decltype(m_)::value + 1;
      constexpr cdouble w = ce_root((long long)j * m, P);
      constexpr float c = float(w.re), sn = float(w.im);
      a = caxpy(c, s[m - 1], a);
      if constexpr (m == 1) b = cscale(sn, d[0]);
      else b = caxpy(sn, d[m - 1], b);
    });
    // x[j] = a + i*DIR*b, x[P-j] = a - i*DIR*b with i*b = (-b.y, b.x)
    constexpr float sg = DIR > 0 ? 1.f : -1.f;
    x[j] = fma2(b.y, b.x, -sg, sg, a.x, a.y);
    x[P - j] = fma2(b.y, b.x, sg, -sg, a.x, a.y);
  });
}

MVD_CE int radix_of(int n) {
  if (n % 4 == 0) return 4;
  if (n % 2 == 0) return 2;
  if (n % 3 == 0) return 3;
  if (n % 5 == 0) return 5;
  if (n % 7 == 0) return 7;
  return n;   // unsupported prime: caught by the static_assert below
}

template <int P, int DIR>
MVD_DEV void bfly(float2 (&t)[P]) {
  static_assert(P == 2 || P == 3 || P == 4 || P == 5 || P == 7, "unsupported radix");
  if constexpr (P == 2) bfly2<DIR>(t[0], t[1]);
  else if constexpr (P == 4) bfly4<DIR>(t[0], t[1], t[2], t[3]);
  else bfly_odd<P, DIR>(t);
}

// ---------------------------------------------------------------------------------------
// N-point DFT in registers:  x[k] <- sum_n x[n] exp(DIR*2*pi*i*n*k/N), natural order in and out.
// Decimation in time with radix P = radix_of(N): P interleaved sub-transforms of length Q = N/P,
// twiddle by W_N^{p k}, then Q radix-P butterflies.
// ---------------------------------------------------------------------------------------
template <int N, int DIR>
struct FftReg {
  static MVD_DEV void run(float2 (&x)[N]) {
#ifdef MVD_SKIP_MATH
    return;
#endif
    if constexpr (N == 1) {
      return;
    } else {
      constexpr int P = radix_of(N);
      constexpr int Q = N / P;
      if constexpr (Q == 1) {
        bfly<P, DIR>(x);
      } else {
        float2 y[P][Q];
        static_for<0, P>([&](auto p_) {
          constexpr int p = decltype(p_)::value;
          static_for<0, Q>([&](auto q_) {
            constexpr int q = decltype(q_)::value;
            y[p][q] = x[q * P + p];
          });
          FftReg<Q, DIR>::run(y[p]);
        });
        static_for<0, Q>([&](auto k_) {
          constexpr int k = decltype(k_)::value;
          float2 t[P];
          static_for<0, P>([&](auto p_) {
            constexpr int p = decltype(p_)::value;
            t[p] = cmul_root<p * k, N, DIR>(y[p][k]);
          });
          bfly<P, DIR>(t);
          static_for<0, P>([&](auto j_) {
            constexpr int j = decltype(j_)::value;
            x[k + Q * j] = t[j];
          });
        });
      }
    }
  }
};

}  // namespace mvd
