// bfly.cuh -- complex fp32 helpers and the radix-2/3/4/5/7 butterflies in registers, shared by the generic tile
// kernel (kernels_generic.cu) and the smooth-digit kernel (smooth.cu).  DIR = +1: exp(-2 pi i pc/r), DIR = -1: exp(+...).
#pragma once
#include <cuda_runtime.h>

namespace dop {

__device__ __forceinline__ float2 cmul(float2 a, float2 b)
{
    return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ float2 cmulc(float2 a, float2 b) // a * conj(b)
{
    return make_float2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }

// one radix-r butterfly, DIR = +1: exp(-2 pi i pc/r), DIR = -1: exp(+...)
template <int DIR>
__device__ __forceinline__ void bfly2(float2* v)
{
    float2 a = v[0], b = v[1];
    v[0] = cadd(a, b);
    v[1] = csub(a, b);
}
template <int DIR>
__device__ __forceinline__ void bfly3(float2* v)
{
    const float h = 0.86602540378443864676f; // sqrt(3)/2
    float2 a = v[0], b = v[1], c = v[2];
    float2 t1 = cadd(b, c);
    float2 t2 = make_float2(a.x - 0.5f * t1.x, a.y - 0.5f * t1.y);
    float2 d = csub(b, c);
    float2 t3 = make_float2(h * d.x, h * d.y);
    v[0] = cadd(a, t1);
    // forward: y1 = t2 - i t3, y2 = t2 + i t3 ; inverse swaps them
    float2 m = make_float2(t2.x + t3.y, t2.y - t3.x); // t2 - i t3
    float2 q = make_float2(t2.x - t3.y, t2.y + t3.x); // t2 + i t3
    if (DIR > 0) { v[1] = m; v[2] = q; } else { v[1] = q; v[2] = m; }
}
template <int DIR>
__device__ __forceinline__ void bfly4(float2* v)
{
    float2 a = v[0], b = v[1], c = v[2], d = v[3];
    float2 s0 = cadd(a, c), s1 = csub(a, c), s2 = cadd(b, d), s3 = csub(b, d);
    v[0] = cadd(s0, s2);
    v[2] = csub(s0, s2);
    float2 m = make_float2(s1.x + s3.y, s1.y - s3.x); // s1 - i s3
    float2 q = make_float2(s1.x - s3.y, s1.y + s3.x); // s1 + i s3
    if (DIR > 0) { v[1] = m; v[3] = q; } else { v[1] = q; v[3] = m; }
}

// radix-5 / radix-7 butterflies in registers: the same symmetric form as prime_step below, unrolled
// (cos / sin of 2 pi k / r as constants).  DIR = +1: exp(-2 pi i pc/r).
template <int DIR>
__device__ __forceinline__ void bfly5(float2* v)
{
    const float c1 = 0.30901699437494742410f, c2 = -0.80901699437494742410f; // cos(2 pi/5), cos(4 pi/5)
    const float s1 = 0.95105651629515357212f, s2 = 0.58778525229247312917f;  // sin(2 pi/5), sin(4 pi/5)
    const float2 a1 = cadd(v[1], v[4]), b1 = csub(v[1], v[4]), a2 = cadd(v[2], v[3]), b2 = csub(v[2], v[3]);
    const float2 x0 = v[0];
    v[0] = cadd(x0, cadd(a1, a2));
    const float2 A1 = make_float2(x0.x + c1 * a1.x + c2 * a2.x, x0.y + c1 * a1.y + c2 * a2.y);
    const float2 A2 = make_float2(x0.x + c2 * a1.x + c1 * a2.x, x0.y + c2 * a1.y + c1 * a2.y);
    const float2 B1 = make_float2(s1 * b1.x + s2 * b2.x, s1 * b1.y + s2 * b2.y);
    const float2 B2 = make_float2(s2 * b1.x - s1 * b2.x, s2 * b1.y - s1 * b2.y);
    // forward: y_k = A_k - i B_k, y_{5-k} = A_k + i B_k
    const float2 m1 = make_float2(A1.x + B1.y, A1.y - B1.x), q1 = make_float2(A1.x - B1.y, A1.y + B1.x);
    const float2 m2 = make_float2(A2.x + B2.y, A2.y - B2.x), q2 = make_float2(A2.x - B2.y, A2.y + B2.x);
    if (DIR > 0) { v[1] = m1; v[4] = q1; v[2] = m2; v[3] = q2; }
    else { v[1] = q1; v[4] = m1; v[2] = q2; v[3] = m2; }
}
template <int DIR>
__device__ __forceinline__ void bfly7(float2* v)
{
    const float c1 = 0.62348980185873353053f, c2 = -0.22252093395631440429f, c3 = -0.90096886790241912624f;
    const float s1 = 0.78183148246802980871f, s2 = 0.97492791218182360702f, s3 = 0.43388373911755812048f;
    const float2 a1 = cadd(v[1], v[6]), b1 = csub(v[1], v[6]), a2 = cadd(v[2], v[5]), b2 = csub(v[2], v[5]);
    const float2 a3 = cadd(v[3], v[4]), b3 = csub(v[3], v[4]);
    const float2 x0 = v[0];
    v[0] = cadd(x0, cadd(a1, cadd(a2, a3)));
    // cos(2 pi c k/7): k=1: c1 c2 c3; k=2: c2 c3 c1; k=3: c3 c1 c2.  sin: k=1: s1 s2 s3; k=2: s2 -s3 -s1; k=3: s3 -s1 s2
    const float2 A1 = make_float2(x0.x + c1 * a1.x + c2 * a2.x + c3 * a3.x, x0.y + c1 * a1.y + c2 * a2.y + c3 * a3.y);
    const float2 A2 = make_float2(x0.x + c2 * a1.x + c3 * a2.x + c1 * a3.x, x0.y + c2 * a1.y + c3 * a2.y + c1 * a3.y);
    const float2 A3 = make_float2(x0.x + c3 * a1.x + c1 * a2.x + c2 * a3.x, x0.y + c3 * a1.y + c1 * a2.y + c2 * a3.y);
    const float2 B1 = make_float2(s1 * b1.x + s2 * b2.x + s3 * b3.x, s1 * b1.y + s2 * b2.y + s3 * b3.y);
    const float2 B2 = make_float2(s2 * b1.x - s3 * b2.x - s1 * b3.x, s2 * b1.y - s3 * b2.y - s1 * b3.y);
    const float2 B3 = make_float2(s3 * b1.x - s1 * b2.x + s2 * b3.x, s3 * b1.y - s1 * b2.y + s2 * b3.y);
    const float2 m1 = make_float2(A1.x + B1.y, A1.y - B1.x), q1 = make_float2(A1.x - B1.y, A1.y + B1.x);
    const float2 m2 = make_float2(A2.x + B2.y, A2.y - B2.x), q2 = make_float2(A2.x - B2.y, A2.y + B2.x);
    const float2 m3 = make_float2(A3.x + B3.y, A3.y - B3.x), q3 = make_float2(A3.x - B3.y, A3.y + B3.x);
    if (DIR > 0) { v[1] = m1; v[6] = q1; v[2] = m2; v[5] = q2; v[3] = m3; v[4] = q3; }
    else { v[1] = q1; v[6] = m1; v[2] = q2; v[5] = m2; v[3] = q3; v[4] = m3; }
}

} // namespace dop
