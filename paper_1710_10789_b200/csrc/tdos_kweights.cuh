// tdos_kweights.cuh -- per-k-point integration weights of the tetrahedron method (Eq. 5-7, :58-71;
// SURVEY.md 8(f) NEXT-2): wk[e][n][k] = sum over the tetrahedra with corner k of w_{n,l}(E_e), so that
// <X>(E_e) = sum_n sum_k X_n(k) wk[e][n][k] for any X (Eq. 7); dwk the same with dw/dE.
//
// The hot path's steps A1-A4 (implicit cubes with periodic wrap, Table I, sort with the permutation, corner
// weights Eq. 11-15) without the orbital projection A5: one thread per (cube, tetrahedron, band), the energies
// taken two at a time with the packed fp32x2 weight routine, results added to the four corner k-points with
// fire-and-forget L2 reductions (each output element receives 24 terms).  Meant for a few energies (a Fermi level,
// a short list), not for a 4000-point grid: the output is nW * nb * nk floats.
#pragma once
#include <cuda_runtime.h>

#include "tdos_kernels.cuh"

namespace tdos {

struct KWeightParams {
    const float* E;
    const float* energies;      // nW energies (device)
    long long sEk, sEn;         // E[ik*sEk + n*sEn]
    int N1, N2, N3, nb, nW;
    float V;                    // V_T/(4 V_G) = 1/(24 nk)
    float* wk;                  // out [nW][nb][nk], zeroed by the caller
    float* dwk;                 // out or null
};

__global__ void __launch_bounds__(256) tdos_kweights(const KWeightParams p) {
    const long long nk = (long long)p.N1 * p.N2 * p.N3;
    const long long total = nk * 6 * p.nb;
    for (long long id = blockIdx.x * (long long)blockDim.x + threadIdx.x; id < total; id += (long long)gridDim.x * blockDim.x) {
        // band slowest, then tetrahedron, cube fastest: neighbouring threads read neighbouring k-points
        const long long cube = id % nk;
        const int tet = (int)((id / nk) % 6), n = (int)(id / (6 * nk));
        const int ix = (int)(cube % p.N1), iy = (int)((cube / p.N1) % p.N2), iz = (int)(cube / ((long long)p.N1 * p.N2));
        float e[4];
        unsigned k[4];
#pragma unroll
        for (int l = 0; l < 4; l++) {
            const int a = kTableI[tet][l];
            const int gx = (ix + (a & 1)) % p.N1, gy = (iy + ((a >> 1) & 1)) % p.N2, gz = (iz + (a >> 2)) % p.N3;
            k[l] = (unsigned)(gx + (long long)p.N1 * (gy + (long long)p.N2 * gz));
            e[l] = __ldg(p.E + (long long)k[l] * p.sEk + (long long)n * p.sEn);
        }
        TDOS_CSWAP(e[0], e[1], k[0], k[1]);
        TDOS_CSWAP(e[2], e[3], k[2], k[3]);
        TDOS_CSWAP(e[0], e[2], k[0], k[2]);
        TDOS_CSWAP(e[1], e[3], k[1], k[3]);
        TDOS_CSWAP(e[1], e[2], k[1], k[2]);
        for (int q = 0; q < p.nW; q += 2) {
            const bool two = q + 1 < p.nW;
            const float Ea = __ldg(p.energies + q), Eb = two ? __ldg(p.energies + q + 1) : Ea;
            f2 w[4], dw[4];
            corner_weights_x2(e[0], e[1], e[2], e[3], make_float2(Ea, Eb), w, dw);   // zero outside (E1, E4)
            // Eq. 15 (test order G10: E <= E1 first, so four equal corners at E give 0)
            const bool fa = Ea >= e[3] && Ea > e[0], fb = Eb >= e[3] && Eb > e[0];
#pragma unroll
            for (int l = 0; l < 4; l++) {
                const float wa = fa ? 1.0f : w[l].x, wb = fb ? 1.0f : w[l].y;
                float* o = p.wk + ((long long)q * p.nb + n) * nk + k[l];
                if (wa != 0.0f) red_add(o, p.V * wa);
                if (two && wb != 0.0f) red_add(o + (long long)p.nb * nk, p.V * wb);
                if (p.dwk) {
                    float* d = p.dwk + ((long long)q * p.nb + n) * nk + k[l];
                    if (dw[l].x != 0.0f) red_add(d, p.V * dw[l].x);
                    if (two && dw[l].y != 0.0f) red_add(d + (long long)p.nb * nk, p.V * dw[l].y);
                }
            }
        }
    }
}

}  // namespace tdos
