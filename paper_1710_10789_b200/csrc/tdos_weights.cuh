// tdos_weights.cuh -- fp32 corner weights of the linear tetrahedron method (device code), evaluated for
// TWO energies at once with Blackwell's packed fp32x2 arithmetic (FFMA2 / FMUL2 / FADD2).
//
// PAPER.md Eq. 11-15 (:105-200), written for the GPU:
//   * every quotient is a product of ratios bounded by 1, so nearly degenerate corners cannot overflow
//     (reading G12); the common factor V = V_T/(4 V_G) is left out (applied once, in fp64, by
//     the finalize kernel);
//   * Eq. 12 and Eq. 14 are mirror images (E - E1 <-> E4 - E, corners 1,2,3,4 <-> 4,3,2,1): one code path
//     ("edge") serves both, its inputs selected per energy;
//   * Eq. 14's weights are formed as w_j = V - C q_j (Eq. 14c/e as printed); only Eq. 15's constant (a finished
//     tetrahedron) is added by the caller as a step at the first energy >= E4;
//   * the derivative identities  sum_l dw_l = 4 dC  (Eq. 12) / -4 dC (Eq. 14)  replace 12d and 14f;
//   * misprints of the paper are read as in DESIGN.md (G1-G5).
// The two energies of a call may fall in different intervals: the edge path and the middle path (Eq. 13)
// each return exact zeros for the energies they do not serve, and the results are added.
//
// This file shares nothing with oracle/ (which restates the same equations literally in fp64).
#pragma once
#include <cuda_runtime.h>

namespace tdos {

typedef float2 f2;
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ f2 add2(f2 a, f2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ f2 dup(float x) { return make_float2(x, x); }

__device__ __forceinline__ float rcp_fast(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// Sorted corner energies e1 <= e2 <= e3 <= e4 and two energies E = (Ea, Eb).
// For each energy with e1 < E < e4:  w[l] = w_l/V,  dw[l] = (dw_l/dE)/V,
// for the sorted corners l = 0..3; for an energy outside (e1, e4), or NaN, all eight values are 0.
__device__ __forceinline__ void corner_weights_x2(float e1, float e2, float e3, float e4, f2 E, f2 (&w)[4], f2 (&dw)[4]) {
    const bool va = (E.x > e1) && (E.x < e4), vb = (E.y > e1) && (E.y < e4);
    const bool lo_a = E.x < e2, lo_b = E.y < e2;          // Eq. 12
    const bool hi_a = E.x >= e3, hi_b = E.y >= e3;        // Eq. 14
    const bool ed_a = va && (lo_a || hi_a), ed_b = vb && (lo_b || hi_b);
    const bool mi_a = va && !lo_a && !hi_a, mi_b = vb && !lo_b && !hi_b;   // Eq. 13

    // reciprocals of the six differences E_ij (Eq. 10); a vanishing difference is never USED by a valid
    // interval (G11), clamping only keeps 0 * (1/0) out of the masked lanes
    const float tiny = 1e-30f;
    const float i21 = rcp_fast(fmaxf(e2 - e1, tiny)), i31 = rcp_fast(fmaxf(e3 - e1, tiny));
    const float i41 = rcp_fast(fmaxf(e4 - e1, tiny)), i32 = rcp_fast(fmaxf(e3 - e2, tiny));
    const float i42 = rcp_fast(fmaxf(e4 - e2, tiny)), i43 = rcp_fast(fmaxf(e4 - e3, tiny));
    const f2 I41 = dup(i41);
    const f2 NEG1 = dup(-1.0f);

#pragma unroll
    for (int l = 0; l < 4; l++) w[l] = dw[l] = dup(0.0f);

    if (ed_a || ed_b) {
        // ---- Eq. 12 / Eq. 14: x = E - E1 (or E4 - E); far corners j: r_j = x/E_j1 (or y/E_4j) <= 1;
        //      C = r r' r'';  w_far = C r_j, dw_far = 4C/E_j1;  w_near = C (4 - sum r), sum_l dw_l = +-4 dC
        f2 X, I1, I2, SG;
        X.x = ed_a ? (lo_a ? E.x - e1 : e4 - E.x) : 0.0f;
        X.y = ed_b ? (lo_b ? E.y - e1 : e4 - E.y) : 0.0f;
        I1.x = lo_a ? i21 : i42;  I1.y = lo_b ? i21 : i42;     // sorted corner 2
        I2.x = lo_a ? i31 : i43;  I2.y = lo_b ? i31 : i43;     // sorted corner 3
        SG.x = lo_a ? 1.0f : -1.0f;  SG.y = lo_b ? 1.0f : -1.0f;   // Eq. 14: w - V = -C q
        const f2 R1 = mul2(X, I1), R2 = mul2(X, I2), R3 = mul2(X, I41);
        const f2 R12 = mul2(R1, R2);
        const f2 C = mul2(R12, R3);                     // 12a / 14a
        const f2 C4 = mul2(C, dup(4.0f));
        const f2 Cs = mul2(C, SG);
        const f2 wF1 = mul2(Cs, R1), wF2 = mul2(Cs, R2), wF3 = mul2(Cs, R3);      // 12e / 14c
        const f2 dF1 = mul2(C4, I1), dF2 = mul2(C4, I2), dF3 = mul2(C4, I41);     // 12f / 14d
        const f2 sumR = add2(add2(R1, R2), R3);
        const f2 wN = fma2(mul2(Cs, NEG1), sumR, mul2(Cs, dup(4.0f)));            // 12c / 14e
        const f2 dN = fma2(mul2(R12, I41), dup(12.0f), mul2(add2(add2(dF1, dF2), dF3), NEG1));   // 12d / 14f
        w[1] = wF1; dw[1] = dF1;
        w[2] = wF2; dw[2] = dF2;
        // the near corner is corner 1 below E2 and corner 4 above E3; the corner with E_41 is the other one
        w[0].x = lo_a ? wN.x : wF3.x;   w[0].y = lo_b ? wN.y : wF3.y;
        w[3].x = lo_a ? wF3.x : wN.x;   w[3].y = lo_b ? wF3.y : wN.y;
        dw[0].x = lo_a ? dN.x : dF3.x;  dw[0].y = lo_b ? dN.y : dF3.y;
        dw[3].x = lo_a ? dF3.x : dN.x;  dw[3].y = lo_b ? dF3.y : dN.y;
        // Eq. 14c/e: w_j = V - C q_j for an energy in [E3, E4)
        const f2 ONE = make_float2((ed_a && !lo_a) ? 1.0f : 0.0f, (ed_b && !lo_b) ? 1.0f : 0.0f);
#pragma unroll
        for (int l = 0; l < 4; l++) w[l] = add2(w[l], ONE);
    }
    if (mi_a || mi_b) {
        // ---- Eq. 13.  For an energy this path does not serve, a = b = 0 makes every term vanish.
        f2 Es, a;
        Es.x = mi_a ? E.x : e2;  Es.y = mi_b ? E.y : e2;
        a.x = mi_a ? Es.x - e1 : 0.0f;  a.y = mi_b ? Es.y - e1 : 0.0f;
        const f2 b = fma2(dup(e2), NEG1, Es);           // E - E2
        const f2 c = fma2(Es, NEG1, dup(e3));           // E3 - E
        const f2 d = fma2(Es, NEG1, dup(e4));           // E4 - E
        const f2 I31 = dup(i31), I32 = dup(i32), I42 = dup(i42);
        const f2 A31 = mul2(a, I31), A41 = mul2(a, I41);     // (E-E1)/E31, (E-E1)/E41
        const f2 B32 = mul2(b, I32), B42 = mul2(b, I42);     // (E-E2)/E32, (E-E2)/E42
        const f2 C31 = mul2(c, I31), C32 = mul2(c, I32);     // (E3-E)/E31, (E3-E)/E32
        const f2 D41 = mul2(d, I41), D42 = mul2(d, I42);     // (E4-E)/E41, (E4-E)/E42
        const f2 C1 = mul2(A31, A41);                                        // 13a
        const f2 dC1 = mul2(A31, dup(2.0f * i41));                           // 13b
        const f2 AB = mul2(A31, B32);
        const f2 C2 = mul2(mul2(A41, B32), C31);                             // 13c
        const f2 dC2 = mul2(I41, fma2(AB, NEG1, mul2(mul2(C32, add2(a, b)), I31)));   // 13d
        const f2 C3 = mul2(mul2(B32, B42), D41);                             // 13e
        const f2 dC3 = mul2(mul2(B32, I41), fma2(B42, NEG1, add2(D42, D42)));   // 13f
        const f2 C12 = add2(C1, C2), C23 = add2(C2, C3), C123 = add2(C12, C3);
        const f2 dC12 = add2(dC1, dC2), dC23 = add2(dC2, dC3), dC123 = add2(dC12, dC3);
        const f2 P = mul2(C12, C31), Q = mul2(C23, C32), R = mul2(C123, D41), S = mul2(C3, D42);
        const f2 dP = fma2(C12, dup(-i31), mul2(dC12, C31));   // d/dE [C12 (E3-E)/E31]
        const f2 dQ = fma2(C23, dup(-i32), mul2(dC23, C32));
        const f2 dR = fma2(C123, dup(-i41), mul2(dC123, D41));
        const f2 dS = fma2(C3, dup(-i42), mul2(dC3, D42));
        w[0] = add2(w[0], add2(add2(C1, P), R));                             // 13g
        w[1] = add2(w[1], add2(add2(C123, Q), S));                           // 13i
        w[2] = add2(w[2], add2(fma2(P, NEG1, C12), fma2(Q, NEG1, C23)));     // 13k (G3): (E-E1)/E31 = 1 - (E3-E)/E31
        w[3] = add2(w[3], add2(fma2(R, NEG1, C123), fma2(S, NEG1, C3)));     // 13m
        dw[0] = add2(dw[0], add2(add2(dC1, dP), dR));                        // 13h
        dw[1] = add2(dw[1], add2(add2(dC123, dQ), dS));                      // 13j
        dw[2] = add2(dw[2], add2(fma2(dP, NEG1, dC12), fma2(dQ, NEG1, dC23)));   // 13l (G4)
        dw[3] = add2(dw[3], add2(fma2(dR, NEG1, dC123), fma2(dS, NEG1, dC3)));   // 13n
    }
}

// The same weights in double precision for ONE energy (TDOS_ACC_FP64_ALL; "one can in principle switch to
// double precision"): the algebra of corner_weights_x2 line by line -- bounded ratios, mirror image for Eq. 14,
// derivative identities -- with true divisions instead of rcp.approx.  w[l] = w_l/V, dw[l] = (dw_l/dE)/V for the
// sorted corners; all zero for an energy outside (e1, e4).  Eq. 15's constant is the caller's step histogram.
__device__ __forceinline__ void corner_weights_f64(double e1, double e2, double e3, double e4, double E, double (&w)[4],
                                                   double (&dw)[4]) {
#pragma unroll
    for (int l = 0; l < 4; l++) w[l] = dw[l] = 0.0;
    if (!((E > e1) && (E < e4))) return;
    const bool lo = E < e2, hi = E >= e3;
    if (lo || hi) {
        // Eq. 12 / Eq. 14: x = E - E1 (or E4 - E); far corners j: r_j = x/E_j1 (or x/E_4j) <= 1; C = r r' r''
        const double x = lo ? E - e1 : e4 - E;
        const double i1 = 1.0 / (lo ? e2 - e1 : e4 - e2);      // sorted corner 2
        const double i2 = 1.0 / (lo ? e3 - e1 : e4 - e3);      // sorted corner 3
        const double i3 = 1.0 / (e4 - e1);                     // the other outer corner
        const double r1 = x * i1, r2 = x * i2, r3 = x * i3;
        const double C = r1 * r2 * r3;                         // 12a / 14a
        const double sg = lo ? 1.0 : -1.0;                     // Eq. 14: w - V = -C q
        const double wF1 = sg * C * r1, wF2 = sg * C * r2, wF3 = sg * C * r3;      // 12e / 14c
        const double dF1 = 4.0 * C * i1, dF2 = 4.0 * C * i2, dF3 = 4.0 * C * i3;   // 12f / 14d
        const double wN = sg * C * (4.0 - (r1 + r2 + r3));                         // 12c / 14e
        const double dN = 12.0 * r1 * r2 * i3 - (dF1 + dF2 + dF3);                 // 12d / 14f: sum_l dw_l = +-4 dC
        const double one = lo ? 0.0 : 1.0;                     // Eq. 14c/e: w_j = V - C q_j
        w[1] = wF1 + one;  dw[1] = dF1;
        w[2] = wF2 + one;  dw[2] = dF2;
        w[0] = (lo ? wN : wF3) + one;  dw[0] = lo ? dN : dF3;
        w[3] = (lo ? wF3 : wN) + one;  dw[3] = lo ? dF3 : dN;
        return;
    }
    // Eq. 13 (e2 <= E < e3; then e3 > e2, e3 > e1, e4 > e2, e4 > e1: no vanishing denominator)
    const double i31 = 1.0 / (e3 - e1), i41 = 1.0 / (e4 - e1), i32 = 1.0 / (e3 - e2), i42 = 1.0 / (e4 - e2);
    const double a = E - e1, b = E - e2, c = e3 - E, d = e4 - E;
    const double A31 = a * i31, A41 = a * i41, B32 = b * i32, B42 = b * i42;
    const double C31 = c * i31, C32 = c * i32, D41 = d * i41, D42 = d * i42;
    const double C1 = A31 * A41;                                        // 13a
    const double dC1 = 2.0 * A31 * i41;                                 // 13b
    const double C2 = A41 * B32 * C31;                                  // 13c
    const double dC2 = i41 * (C32 * (a + b) * i31 - A31 * B32);         // 13d
    const double C3 = B32 * B42 * D41;                                  // 13e
    const double dC3 = B32 * i41 * (2.0 * D42 - B42);                   // 13f
    const double C12 = C1 + C2, C23 = C2 + C3, C123 = C12 + C3;
    const double dC12 = dC1 + dC2, dC23 = dC2 + dC3, dC123 = dC12 + dC3;
    const double P = C12 * C31, Q = C23 * C32, R = C123 * D41, S = C3 * D42;
    const double dP = dC12 * C31 - C12 * i31, dQ = dC23 * C32 - C23 * i32;
    const double dR = dC123 * D41 - C123 * i41, dS = dC3 * D42 - C3 * i42;
    w[0] = C1 + P + R;                  dw[0] = dC1 + dP + dR;                    // 13g, 13h
    w[1] = C123 + Q + S;                dw[1] = dC123 + dQ + dS;                  // 13i, 13j
    w[2] = (C12 - P) + (C23 - Q);       dw[2] = (dC12 - dP) + (dC23 - dQ);        // 13k (G3), 13l (G4)
    w[3] = (C123 - R) + (C3 - S);       dw[3] = (dC123 - dR) + (dC3 - dS);        // 13m, 13n
}

}  // namespace tdos
