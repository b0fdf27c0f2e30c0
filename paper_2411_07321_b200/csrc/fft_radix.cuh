// fft_radix.cuh -- small inverse DFTs (sign +, un-normalised: D7) on register arrays, for float2 and double2.
// Used by the split column transform (colsplit.cu).  Nothing here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>

#define RICK_DI __device__ __forceinline__

template <typename C2> struct RickRealOf;
template <> struct RickRealOf<float2> { typedef float type; };
template <> struct RickRealOf<double2> { typedef double type; };

template <typename C2> RICK_DI C2 cx_make(typename RickRealOf<C2>::type x, typename RickRealOf<C2>::type y) {
    C2 r;
    r.x = x;
    r.y = y;
    return r;
}
// double2 (and the generic fallback): scalar arithmetic
template <typename C2> RICK_DI C2 cx_add(C2 a, C2 b) { return cx_make<C2>(a.x + b.x, a.y + b.y); }
template <typename C2> RICK_DI C2 cx_sub(C2 a, C2 b) { return cx_make<C2>(a.x - b.x, a.y - b.y); }
template <typename C2> RICK_DI C2 cx_mul(C2 a, C2 b) { return cx_make<C2>(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
template <typename C2> RICK_DI C2 cx_mul_i(C2 a) { return cx_make<C2>(-a.y, a.x); }      // a * i
template <typename C2> RICK_DI C2 cx_scale(typename RickRealOf<C2>::type r, C2 a) { return cx_make<C2>(r * a.x, r * a.y); }

// float2: the packed fp32 instructions of sm_100 (add / sub / mul / fma .f32x2 -> SASS FADD2 / FMUL2 / FFMA2, one
// issue slot for the (re, im) pair; the half swap and the negations of "times i" are operand modifiers)
RICK_DI unsigned long long cx_pack(float x, float y) {
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(x), "f"(y));
    return r;
}
RICK_DI float2 cx_unpack(unsigned long long a) {
    float2 r;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(a));
    return r;
}
template <> RICK_DI float2 cx_add<float2>(float2 a, float2 b) {
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(cx_pack(a.x, a.y)), "l"(cx_pack(b.x, b.y)));
    return cx_unpack(r);
}
template <> RICK_DI float2 cx_sub<float2>(float2 a, float2 b) {
    unsigned long long r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(cx_pack(a.x, a.y)), "l"(cx_pack(b.x, b.y)));
    return cx_unpack(r);
}
template <> RICK_DI float2 cx_scale<float2>(float r, float2 a) {
    unsigned long long o;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(o) : "l"(cx_pack(r, r)), "l"(cx_pack(a.x, a.y)));
    return cx_unpack(o);
}
// (a.x b.x - a.y b.y, a.x b.y + a.y b.x) = (a.x, a.x) * b + (a.y, a.y) * (-b.y, b.x)
template <> RICK_DI float2 cx_mul<float2>(float2 a, float2 b) {
    unsigned long long t, o;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(t) : "l"(cx_pack(a.y, a.y)), "l"(cx_pack(-b.y, b.x)));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(o) : "l"(cx_pack(a.x, a.x)), "l"(cx_pack(b.x, b.y)), "l"(t));
    return cx_unpack(o);
}
// acc + s * v for a real s (both halves): the gridder's accumulation and the screen-free twiddle products
RICK_DI float2 cx_fma_real(float s, float2 v, float2 acc) {
    unsigned long long o;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(o) : "l"(cx_pack(s, s)), "l"(cx_pack(v.x, v.y)), "l"(cx_pack(acc.x, acc.y)));
    return cx_unpack(o);
}

// 4-point inverse DFT (omega_4 = +i), natural order in and out
template <typename C2> RICK_DI void cx_dft4(C2& a, C2& b, C2& c, C2& d) {
    const C2 s0 = cx_add(a, c), d0 = cx_sub(a, c), s1 = cx_add(b, d), d1 = cx_sub(b, d);
    a = cx_add(s0, s1);
    c = cx_sub(s0, s1);
    const C2 id1 = cx_mul_i(d1);
    b = cx_add(d0, id1);                            // d0 + i d1
    d = cx_sub(d0, id1);                            // d0 - i d1
}

// R-point inverse DFT, y_u = sum_t x_t exp(+2 pi i u t / R), natural order in and out, R in {1, 2, 4, 8, 16}
template <int R, typename C2> RICK_DI void cx_dft(C2* v) {
    typedef typename RickRealOf<C2>::type real;
    if constexpr (R == 2) {
        const C2 a = v[0], b = v[1];
        v[0] = cx_add(a, b);
        v[1] = cx_sub(a, b);
    } else if constexpr (R == 4) {
        cx_dft4(v[0], v[1], v[2], v[3]);
    } else if constexpr (R == 8) {
        C2 e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6], o0 = v[1], o1 = v[3], o2 = v[5], o3 = v[7];
        cx_dft4(e0, e1, e2, e3);
        cx_dft4(o0, o1, o2, o3);
        const real r = (real)0.70710678118654752440;
        const C2 t1 = cx_scale(r, cx_add(o1, cx_mul_i(o1)));      // o1 * exp(+i pi/4)   = r (o1 + i o1)
        const C2 t2 = cx_mul_i(o2);                                 // o2 * i
        const C2 t3 = cx_scale(r, cx_sub(cx_mul_i(o3), o3));      // o3 * exp(+3 i pi/4) = r (i o3 - o3)
        v[0] = cx_add(e0, o0); v[4] = cx_sub(e0, o0);
        v[1] = cx_add(e1, t1); v[5] = cx_sub(e1, t1);
        v[2] = cx_add(e2, t2); v[6] = cx_sub(e2, t2);
        v[3] = cx_add(e3, t3); v[7] = cx_sub(e3, t3);
    } else if constexpr (R == 16) {
        // 16 = 4 x 4: t = 4a + b, u = c + 4d:  w16^(ut) = w4^(ac) w16^(bc) w4^(bd)
#pragma unroll
        for (int b = 0; b < 4; ++b) cx_dft4(v[b], v[4 + b], v[8 + b], v[12 + b]);   // over a: result c at v[4c + b]
        const real c1 = (real)0.92387953251128675613, s1 = (real)0.38268343236508977173, r = (real)0.70710678118654752440;
        const C2 w1 = cx_make<C2>(c1, s1), w3 = cx_make<C2>(s1, c1), w9 = cx_make<C2>(-c1, -s1);
        // w2 = r (1 + i): v w2 = r (v + i v);  w6 = r (-1 + i): v w6 = r (i v - v)
        v[4 + 1] = cx_mul(v[4 + 1], w1); v[4 + 2] = cx_scale(r, cx_add(v[4 + 2], cx_mul_i(v[4 + 2]))); v[4 + 3] = cx_mul(v[4 + 3], w3);
        v[8 + 1] = cx_scale(r, cx_add(v[8 + 1], cx_mul_i(v[8 + 1]))); v[8 + 2] = cx_mul_i(v[8 + 2]);
        v[8 + 3] = cx_scale(r, cx_sub(cx_mul_i(v[8 + 3]), v[8 + 3]));
        v[12 + 1] = cx_mul(v[12 + 1], w3); v[12 + 2] = cx_scale(r, cx_sub(cx_mul_i(v[12 + 2]), v[12 + 2])); v[12 + 3] = cx_mul(v[12 + 3], w9);
#pragma unroll
        for (int c = 0; c < 4; ++c) cx_dft4(v[4 * c], v[4 * c + 1], v[4 * c + 2], v[4 * c + 3]);   // over b: d at v[4c + d]
#pragma unroll
        for (int c = 0; c < 4; ++c)          // y(c + 4d) sits at v[4c + d]: transpose so that y_u is at v[u]
#pragma unroll
            for (int d = c + 1; d < 4; ++d) {
                const C2 t = v[4 * c + d];
                v[4 * c + d] = v[4 * d + c];
                v[4 * d + c] = t;
            }
    }
}
