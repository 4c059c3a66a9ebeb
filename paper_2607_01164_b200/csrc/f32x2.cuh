// f32x2.cuh -- packed FP32 arithmetic of sm_100 (fma / mul / add / sub .rn.f32x2 = FFMA2 / FMUL2 / FADD2).
// One lane-instruction does the operation on both halves of a 64-bit register pair; each half is rounded to nearest
// exactly like the scalar instruction, so the canonical predicate sequence (DESIGN D4) keeps its bits when two samples
// (or two Gaussians) ride in the two halves.  The FMA pipe retires the same number of FMAs per clock either way (the
// micro-benchmark of peaks.cu measures 35.9 T lane-operations/s packed against 35.3 T scalar): what the packed form
// saves is ISSUE SLOTS, which is what the sampling kernels are short of (70-85 % issue utilisation at 36-51 % FMA pipe).
// A scalar that multiplies both halves costs nothing: ptxas folds pk(s, s) into the operand modifier `R.F32`.
// ptxas contracts mul.rn.f32x2 + add.rn.f32x2 into one FFMA2 (it does not for the scalar .rn forms): nothing that feeds
// an integer decision may be written as a packed mul followed by a packed add of its result.  The canonical sequence
// has no such pair (its products are the ADDENDS of the following fma).
#pragma once
#include <cuda_runtime.h>

namespace gs {

typedef unsigned long long f2;  // two floats: .x = low half, .y = high half

__device__ __forceinline__ f2 pk(float lo, float hi) {
    f2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ f2 bc(float s) { return pk(s, s); }  // both halves = s (free: operand modifier .F32)
__device__ __forceinline__ void upk(f2 v, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ float lo(f2 v) { float a, b; upk(v, a, b); return a; }
__device__ __forceinline__ float hi(f2 v) { float a, b; upk(v, a, b); return b; }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) {
    f2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f2 mul2(f2 a, f2 b) {
    f2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f2 add2(f2 a, f2 b) {
    f2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f2 sub2(f2 a, f2 b) {
    f2 d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

// The canonical sequence (D4) for TWO samples against one Gaussian (mu, rows of M as scalars):
//   d = p - mu;  u_j = fma(M_j2, dz, fma(M_j1, dy, M_j0 * dx));  qd = fma(u2, u2, fma(u1, u1, u0 * u0))
// Each packed instruction performs the scalar operation of the sequence on both halves.
__device__ __forceinline__ f2 mahalanobis2(float mx, float my, float mz, float m00, float m01, float m02, float m10, float m11,
                                           float m12, float m20, float m21, float m22, f2 px, f2 py, f2 pz, f2 &u0, f2 &u1, f2 &u2) {
    const f2 dx = sub2(px, bc(mx)), dy = sub2(py, bc(my)), dz = sub2(pz, bc(mz));
    u0 = fma2(bc(m02), dz, fma2(bc(m01), dy, mul2(bc(m00), dx)));
    u1 = fma2(bc(m12), dz, fma2(bc(m11), dy, mul2(bc(m10), dx)));
    u2 = fma2(bc(m22), dz, fma2(bc(m21), dy, mul2(bc(m20), dx)));
    return fma2(u2, u2, fma2(u1, u1, mul2(u0, u0)));
}

// G = exp(-qd / 2) for the halves that pass the canonical predicate qd <= r2, 0 for the others (value arithmetic).
__device__ __forceinline__ f2 gauss_weight2(f2 qd, float r2, bool &hit_lo, bool &hit_hi) {
    float qa, qb, ta, tb, ga, gb;
    upk(qd, qa, qb);
    upk(mul2(qd, bc(-0.72134752044448170368f)), ta, tb);
    hit_lo = qa <= r2;
    hit_hi = qb <= r2;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(ga) : "f"(ta));
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(gb) : "f"(tb));
    return pk(hit_lo ? ga : 0.f, hit_hi ? gb : 0.f);
}

}  // namespace gs
