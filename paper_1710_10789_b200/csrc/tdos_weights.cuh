// tdos_weights.cuh -- fp32 corner weights of the linear tetrahedron method (device code).
//
// PAPER.md Eq. 11-15 (:105-200), written for the GPU: every quotient is formed as a product of
// ratios bounded by 1 (so nearly degenerate corners cannot overflow, reading G12), the
// common factor V = V_T/(4 V_G) is left out (applied once, in fp64, by the merge kernel), and the
// derivative identities  sum_l dw_l = 4 dC  (Eq. 12) /  -4 dC (Eq. 14)  replace the longest
// expressions (12d, 14f).  Misprints of the paper are read as in DESIGN.md (G1-G5).
//
// This file shares nothing with oracle/ (which restates the same equations literally in fp64).
#pragma once
#include <cuda_runtime.h>

namespace tdos {

__device__ __forceinline__ float rcp_fast(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// Sorted corner energies e1 <= e2 <= e3 <= e4, energy of interest E with e1 < E < e4.
// Outputs w[l]/V and (dw[l]/dE)/V for the sorted corners l = 0..3.
__device__ __forceinline__ void corner_weights_in_window(float e1, float e2, float e3, float e4, float E,
                                                         float (&w)[4], float (&dw)[4]) {
    if (E < e2) {
        // Eq. 12: x = E - E1, r_j = x/E_j1 <= 1, C = r2 r3 r4
        const float x = E - e1;
        const float i21 = rcp_fast(e2 - e1), i31 = rcp_fast(e3 - e1), i41 = rcp_fast(e4 - e1);
        const float r2 = x * i21, r3 = x * i31, r4 = x * i41;
        const float r23 = r2 * r3;
        const float C = r23 * r4;                  // 12a
        const float dC = 3.0f * r23 * i41;         // 12b
        const float C4 = 4.0f * C;
        w[1] = C * r2;                             // 12e
        w[2] = C * r3;
        w[3] = C * r4;
        w[0] = fmaf(-C, (r2 + r3) + r4, C4);       // 12c
        dw[1] = C4 * i21;                          // 12f: dC x/E_j1 + C/E_j1 = 4C/E_j1
        dw[2] = C4 * i31;
        dw[3] = C4 * i41;
        dw[0] = fmaf(4.0f, dC, -((dw[1] + dw[2]) + dw[3]));   // 12d via sum_l dw_l = 4 dC
    } else if (E < e3) {
        // Eq. 13
        const float a = E - e1, b = E - e2, c = e3 - E, d = e4 - E;
        const float i31 = rcp_fast(e3 - e1), i41 = rcp_fast(e4 - e1);
        const float i32 = rcp_fast(e3 - e2), i42 = rcp_fast(e4 - e2);
        const float A31 = a * i31, A41 = a * i41;  // (E-E1)/E31, (E-E1)/E41
        const float B32 = b * i32, B42 = b * i42;  // (E-E2)/E32, (E-E2)/E42
        const float C31 = c * i31, C32 = c * i32;  // (E3-E)/E31, (E3-E)/E32
        const float D41 = d * i41, D42 = d * i42;  // (E4-E)/E41, (E4-E)/E42
        const float C1 = A31 * A41;                                        // 13a
        const float dC1 = 2.0f * A31 * i41;                                // 13b
        const float AB = A31 * B32;
        const float C2 = A41 * B32 * C31;                                  // 13c
        const float dC2 = i41 * fmaf(C32 * (a + b), i31, -AB);             // 13d
        const float BB = B32 * B42;
        const float C3 = BB * D41;                                         // 13e
        const float dC3 = B32 * i41 * fmaf(2.0f, D42, -B42);               // 13f
        const float C12 = C1 + C2, C23 = C2 + C3, C123 = C12 + C3;
        const float dC12 = dC1 + dC2, dC23 = dC2 + dC3, dC123 = dC12 + dC3;
        const float P = C12 * C31, Q = C23 * C32, R = C123 * D41, S = C3 * D42;
        w[0] = (C1 + P) + R;                                               // 13g
        w[1] = (C123 + Q) + S;                                             // 13i
        w[2] = (C12 - P) + (C23 - Q);                                      // 13k (G3): (E-E1)/E31 = 1 - (E3-E)/E31
        w[3] = (C123 - R) + (C3 - S);                                      // 13m
        const float dP = fmaf(dC12, C31, -C12 * i31);    // d/dE [C12 (E3-E)/E31]
        const float dQ = fmaf(dC23, C32, -C23 * i32);
        const float dR = fmaf(dC123, D41, -C123 * i41);
        const float dS = fmaf(dC3, D42, -C3 * i42);
        dw[0] = (dC1 + dP) + dR;                                           // 13h
        dw[1] = (dC123 + dQ) + dS;                                         // 13j
        dw[2] = (dC12 - dP) + (dC23 - dQ);                                 // 13l (G4)
        dw[3] = (dC123 - dR) + (dC3 - dS);                                 // 13n
    } else {
        // Eq. 14: y = E4 - E, q_j = y/E_4j <= 1, C = q1 q2 q3
        const float y = e4 - E;
        const float i41 = rcp_fast(e4 - e1), i42 = rcp_fast(e4 - e2), i43 = rcp_fast(e4 - e3);
        const float q1 = y * i41, q2 = y * i42, q3 = y * i43;
        const float q12 = q1 * q2;
        const float C = q12 * q3;                  // 14a
        const float mdC = 3.0f * q12 * i43;        // -(14b)
        const float C4 = 4.0f * C;
        w[0] = fmaf(-C, q1, 1.0f);                 // 14c
        w[1] = fmaf(-C, q2, 1.0f);
        w[2] = fmaf(-C, q3, 1.0f);
        w[3] = 1.0f - fmaf(-C, (q1 + q2) + q3, C4);    // 14e (G5)
        dw[0] = C4 * i41;                          // 14d: -dC y/E_4j + C/E_4j = 4C/E_4j
        dw[1] = C4 * i42;
        dw[2] = C4 * i43;
        dw[3] = fmaf(4.0f, mdC, -((dw[0] + dw[1]) + dw[2]));   // 14f via sum_l dw_l = -4 dC
    }
}

}  // namespace tdos
