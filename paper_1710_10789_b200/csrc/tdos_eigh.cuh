// tdos_eigh.cuh -- batched Hermitian eigensolver for the input side of the path:
// PAPER.md Eq. 1 (:37-39) "diagonalised to obtain band energies E_n(k) and eigenvector elements a_n^m(k)", so that
// H(k) -> E, a -> DOS never leaves the device (the paper's "best case": "input data naturally reside in GPU memory", :289).
//
// Cyclic Jacobi method for complex Hermitian matrices of order <= 8, 8 lanes per matrix (4 matrices per warp):
// lane r keeps row r of H and row r of the eigenvector matrix V (V[m][n] = a_n^m) in registers.  A sweep is the 7
// rounds of a round-robin tournament; a round rotates 4 disjoint pairs (p, q) at once:
//     J = [[c, s], [-s e^{-i phi}, c e^{-i phi}]],  H_pq = |H_pq| e^{i phi},  t = s/c the smaller root of t^2 + 2 tau t - 1 = 0,
//     tau = (H_qq - H_pp) / (2 |H_pq|),     H <- J^H H J,   V <- V J.
// The pairs of a round are compile-time constants (fully unrolled), so all register indices are static; the column
// part of H <- J^H (H J) and V <- V J is local to a lane, the row part is one exchange of rows between the two lanes
// of a pair (shuffles).  The arithmetic is fp64 (as the host LAPACK call it replaces; the results are rounded to the
// fp32 arrays the path consumes).  Sweeps stop when every matrix of the warp has an off-diagonal Frobenius norm below
// 1e-12 of its own norm, at most `sweeps` (10) of them (the method converges quadratically; 4-6 are typical for
// order 8).  Only the upper triangle of H is read.  Eigenvalues are written in ascending order with their eigenvectors.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tdos {

struct EighParams {
    const float2* H;     // [nmat][nb][nb] row-major, Hermitian
    float* E;            // [nmat][nb] ascending
    float2* A;           // [nmat][nb][nb]: A[i][n][m] = component m of eigenvector n
    long long nmat;
    int nb;              // 1..8 (tdos_eigh8), 9..16 (tdos_eigh_n<16>)
    int sweeps;
};

// round-robin tournament on 8 players: round s (0..6), pair k (0..3) -> (p, q)
__host__ __device__ constexpr int rr_player(int s, int pos) {   // pos 0 is fixed, positions 1..7 rotate
    return pos == 0 ? 0 : 1 + (pos - 1 + s) % 7;
}
__host__ __device__ constexpr int rr_p(int s, int k) { return k == 0 ? rr_player(s, 0) : rr_player(s, k); }
__host__ __device__ constexpr int rr_q(int s, int k) { return k == 0 ? rr_player(s, 7) : rr_player(s, 7 - k); }

template <int S>
__device__ __forceinline__ void jacobi_round(double (&hr)[8], double (&hi)[8], double (&vr)[8], double (&vi)[8], int r, int base,
                                             unsigned mask) {
    // parameters of the 4 rotations, computed by every lane from broadcast matrix elements
    double c[4], s[4], er[4], ei[4];   // e = e^{i phi}
#pragma unroll
    for (int k = 0; k < 4; k++) {
        const int p = rr_p(S, k), q = rr_q(S, k);
        const double a = __shfl_sync(mask, hr[p], base + p);     // H_pp (lane p, column p)
        const double b = __shfl_sync(mask, hr[q], base + q);     // H_qq
        const double gr = __shfl_sync(mask, hr[q], base + p);    // H_pq (lane p, column q)
        const double gi = __shfl_sync(mask, hi[q], base + p);
        const double g2 = gr * gr + gi * gi;
        if (g2 > 1e-280) {
            const double ig = 1.0 / sqrt(g2);
            const double tau = (b - a) * (0.5 * ig);
            const double t = copysign(1.0, tau) / (fabs(tau) + sqrt(1.0 + tau * tau));
            c[k] = 1.0 / sqrt(1.0 + t * t);
            s[k] = t * c[k];
            er[k] = gr * ig;
            ei[k] = gi * ig;
        } else {
            c[k] = 1.0; s[k] = 0.0; er[k] = 1.0; ei[k] = 0.0;
        }
    }
    // columns: X[:, p'] = c X[:, p] - s e^{-i phi} X[:, q],  X[:, q'] = s X[:, p] + c e^{-i phi} X[:, q]   (X = H, V)
#pragma unroll
    for (int k = 0; k < 4; k++) {
        const int p = rr_p(S, k), q = rr_q(S, k);
        {
            const double xr = hr[p], xi = hi[p];
            const double yr = hr[q] * er[k] + hi[q] * ei[k], yi = hi[q] * er[k] - hr[q] * ei[k];   // e^{-i phi} X_q
            hr[p] = c[k] * xr - s[k] * yr; hi[p] = c[k] * xi - s[k] * yi;
            hr[q] = s[k] * xr + c[k] * yr; hi[q] = s[k] * xi + c[k] * yi;
        }
        {
            const double xr = vr[p], xi = vi[p];
            const double yr = vr[q] * er[k] + vi[q] * ei[k], yi = vi[q] * er[k] - vr[q] * ei[k];
            vr[p] = c[k] * xr - s[k] * yr; vi[p] = c[k] * xi - s[k] * yi;
            vr[q] = s[k] * xr + c[k] * yr; vi[q] = s[k] * xi + c[k] * yi;
        }
    }
    // rows of H: X[p', :] = c X[p, :] - s e^{+i phi} X[q, :],  X[q', :] = s X[p, :] + c e^{+i phi} X[q, :]
    int partner = r, kk = 0;
    bool is_p = true;
#pragma unroll
    for (int k = 0; k < 4; k++) {
        const int p = rr_p(S, k), q = rr_q(S, k);
        if (r == p) { partner = q; kk = k; is_p = true; }
        if (r == q) { partner = p; kk = k; is_p = false; }
    }
    const double cc = kk == 0 ? c[0] : kk == 1 ? c[1] : kk == 2 ? c[2] : c[3];
    const double ss = kk == 0 ? s[0] : kk == 1 ? s[1] : kk == 2 ? s[2] : s[3];
    const double fr = kk == 0 ? er[0] : kk == 1 ? er[1] : kk == 2 ? er[2] : er[3];
    const double fi = kk == 0 ? ei[0] : kk == 1 ? ei[1] : kk == 2 ? ei[2] : ei[3];
#pragma unroll
    for (int j = 0; j < 8; j++) {
        const double tr = __shfl_sync(mask, hr[j], base + partner), ti = __shfl_sync(mask, hi[j], base + partner);
        // row p (mine) and row q (theirs) if is_p, else the other way round
        const double pr = is_p ? hr[j] : tr, pi = is_p ? hi[j] : ti;
        const double qr0 = is_p ? tr : hr[j], qi0 = is_p ? ti : hi[j];
        const double qr = qr0 * fr - qi0 * fi, qi = qr0 * fi + qi0 * fr;   // e^{+i phi} X_q
        hr[j] = is_p ? cc * pr - ss * qr : ss * pr + cc * qr;
        hi[j] = is_p ? cc * pi - ss * qi : ss * pi + cc * qi;
    }
}

__global__ void __launch_bounds__(128, 4) tdos_eigh8(const EighParams P) {
    const int lane = threadIdx.x & 31, r = lane & 7, base = lane & ~7;
    const long long mat = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 3;
    const bool live = mat < P.nmat;
    const unsigned mask = 0xffffffffu;
    const int nb = P.nb;
    double hr[8], hi[8], vr[8], vi[8];
#pragma unroll
    for (int j = 0; j < 8; j++) {
        hr[j] = (j == r && r >= nb) ? 1e30 * (1 + r) : 0.0;   // padding: decoupled levels far above, sorted last
        hi[j] = 0.0;
        vr[j] = (j == r) ? 1.0 : 0.0;
        vi[j] = 0.0;
    }
    // Only the upper triangle of the input is read: H_rj for j >= r, its conjugate for j < r, a real diagonal.  An input
    // that is Hermitian only to fp32 rounding (assembled on the device) is thereby made exactly Hermitian, which the
    // rotations below rely on (they read H_pq from row p and never look at H_qp).
    if (live && r < nb) {
        const float2* M = P.H + mat * nb * nb;
#pragma unroll
        for (int j = 0; j < 8; j++)
            if (j < nb) {
                const float2 z = __ldg(j >= r ? M + r * nb + j : M + j * nb + r);
                hr[j] = z.x;
                hi[j] = j > r ? z.y : j < r ? -z.y : 0.0;
            }
    }
    for (int sweep = 0; sweep < P.sweeps; ++sweep) {
        // Convergence: stop once, for every matrix of the warp, the off-diagonal part is below 1e-12 of the matrix in
        // the Frobenius norm (the outputs are rounded to fp32, 6e-8).  Padded rows (r >= nb) count as zero.
        double off = 0.0, all = 0.0;
#pragma unroll
        for (int j = 0; j < 8; j++) {
            const double a2 = (r < nb) ? hr[j] * hr[j] + hi[j] * hi[j] : 0.0;
            all += a2;
            if (j != r) off += a2;
        }
#pragma unroll
        for (int d = 1; d < 8; d <<= 1) {
            off += __shfl_xor_sync(mask, off, d);
            all += __shfl_xor_sync(mask, all, d);
        }
        if (!__any_sync(mask, live && off > 1e-24 * all)) break;
        jacobi_round<0>(hr, hi, vr, vi, r, base, mask);
        jacobi_round<1>(hr, hi, vr, vi, r, base, mask);
        jacobi_round<2>(hr, hi, vr, vi, r, base, mask);
        jacobi_round<3>(hr, hi, vr, vi, r, base, mask);
        jacobi_round<4>(hr, hi, vr, vi, r, base, mask);
        jacobi_round<5>(hr, hi, vr, vi, r, base, mask);
        jacobi_round<6>(hr, hi, vr, vi, r, base, mask);
    }
    // eigenvalue of column c: the diagonal element H_cc (lane c); rank = its place in ascending order (ties by index)
    double lam[8];
#pragma unroll
    for (int c = 0; c < 8; c++) lam[c] = __shfl_sync(mask, hr[c], base + c);
    if (!live) return;
#pragma unroll
    for (int c = 0; c < 8; c++) {
        int rank = 0;
#pragma unroll
        for (int d = 0; d < 8; d++) rank += (lam[d] < lam[c] || (lam[d] == lam[c] && d < c)) ? 1 : 0;
        if (rank < nb && r < nb) {
            if (r == 0) P.E[mat * nb + rank] = (float)lam[c];
            P.A[(mat * nb + rank) * nb + r] = make_float2((float)vr[c], (float)vi[c]);   // component m = r of eigenvector `rank`
        }
    }
}

// ---- orders 9..16 ("16 orbitals correspond to the largest models of iron-based superconductors currently
// considered"): the same method with N = 16 lanes per matrix (2 matrices per warp), N - 1 rounds of N/2 disjoint
// rotations per sweep.  The rotations of a round are taken one after the other (parameters from 4 broadcasts, column
// update of H and V at once), so only one set of rotation parameters is live beside the 4 N doubles of state; a lane
// keeps the parameters of the pair its own row belongs to for the row half.  Disjoint pairs do not touch each other's
// H_pp, H_qq, H_pq, so taking them in sequence gives the same rotations as taking them together.
template <int N>
__host__ __device__ constexpr int rrn_player(int s, int pos) {   // circle method: position 0 fixed, 1..N-1 rotate
    return pos == 0 ? 0 : 1 + (pos - 1 + s) % (N - 1);
}

template <int N, int S>
__device__ __forceinline__ void jacobi_round_n(double (&hr)[N], double (&hi)[N], double (&vr)[N], double (&vi)[N], int r, int base) {
    constexpr unsigned mask = 0xffffffffu;
    double cc = 1.0, ss = 0.0, fr = 1.0, fi = 0.0;
    int partner = r;
    bool is_p = true;
#pragma unroll
    for (int k = 0; k < N / 2; k++) {
        const int p = rrn_player<N>(S, k), q = rrn_player<N>(S, N - 1 - k);
        const double a = __shfl_sync(mask, hr[p], base + p);     // H_pp
        const double b = __shfl_sync(mask, hr[q], base + q);     // H_qq
        const double gr = __shfl_sync(mask, hr[q], base + p);    // H_pq = |H_pq| e^{i phi}
        const double gi = __shfl_sync(mask, hi[q], base + p);
        const double g2 = gr * gr + gi * gi;
        double c = 1.0, s = 0.0, er = 1.0, ei = 0.0;
        if (g2 > 1e-280) {
            const double ig = 1.0 / sqrt(g2);
            const double tau = (b - a) * (0.5 * ig);
            const double t = copysign(1.0, tau) / (fabs(tau) + sqrt(1.0 + tau * tau));
            c = 1.0 / sqrt(1.0 + t * t);
            s = t * c;
            er = gr * ig;
            ei = gi * ig;
        }
        // columns: X[:, p'] = c X[:, p] - s e^{-i phi} X[:, q],  X[:, q'] = s X[:, p] + c e^{-i phi} X[:, q]   (X = H, V)
        {
            const double xr = hr[p], xi = hi[p];
            const double yr = hr[q] * er + hi[q] * ei, yi = hi[q] * er - hr[q] * ei;
            hr[p] = c * xr - s * yr; hi[p] = c * xi - s * yi;
            hr[q] = s * xr + c * yr; hi[q] = s * xi + c * yi;
        }
        {
            const double xr = vr[p], xi = vi[p];
            const double yr = vr[q] * er + vi[q] * ei, yi = vi[q] * er - vr[q] * ei;
            vr[p] = c * xr - s * yr; vi[p] = c * xi - s * yi;
            vr[q] = s * xr + c * yr; vi[q] = s * xi + c * yi;
        }
        if (r == p || r == q) {
            cc = c; ss = s; fr = er; fi = ei;
            partner = (r == p) ? q : p;
            is_p = (r == p);
        }
    }
    // rows of H: X[p', :] = c X[p, :] - s e^{+i phi} X[q, :],  X[q', :] = s X[p, :] + c e^{+i phi} X[q, :]
#pragma unroll
    for (int j = 0; j < N; j++) {
        const double tr = __shfl_sync(mask, hr[j], base + partner), ti = __shfl_sync(mask, hi[j], base + partner);
        const double pr = is_p ? hr[j] : tr, pi = is_p ? hi[j] : ti;
        const double qr0 = is_p ? tr : hr[j], qi0 = is_p ? ti : hi[j];
        const double qr = qr0 * fr - qi0 * fi, qi = qr0 * fi + qi0 * fr;
        hr[j] = is_p ? cc * pr - ss * qr : ss * pr + cc * qr;
        hi[j] = is_p ? cc * pi - ss * qi : ss * pi + cc * qi;
    }
}

template <int N, int S>
struct JacobiSweep {
    static __device__ __forceinline__ void run(double (&hr)[N], double (&hi)[N], double (&vr)[N], double (&vi)[N], int r, int base) {
        jacobi_round_n<N, S>(hr, hi, vr, vi, r, base);
        JacobiSweep<N, S + 1>::run(hr, hi, vr, vi, r, base);
    }
};
template <int N>
struct JacobiSweep<N, N - 1> {
    static __device__ __forceinline__ void run(double (&)[N], double (&)[N], double (&)[N], double (&)[N], int, int) {}
};

template <int N>
__global__ void __launch_bounds__(128) tdos_eigh_n(const EighParams P) {
    static_assert(N == 16, "lanes per matrix");
    const int lane = threadIdx.x & 31, r = lane & (N - 1), base = lane & ~(N - 1);
    const long long mat = (blockIdx.x * (long long)blockDim.x + threadIdx.x) / N;
    const bool live = mat < P.nmat;
    const unsigned mask = 0xffffffffu;
    const int nb = P.nb;
    double hr[N], hi[N], vr[N], vi[N];
#pragma unroll
    for (int j = 0; j < N; j++) {
        hr[j] = (j == r && r >= nb) ? 1e30 * (1 + r) : 0.0;   // padding: decoupled levels far above, sorted last
        hi[j] = 0.0;
        vr[j] = (j == r) ? 1.0 : 0.0;
        vi[j] = 0.0;
    }
    if (live && r < nb) {   // upper triangle only, mirrored (see tdos_eigh8)
        const float2* M = P.H + mat * nb * nb;
#pragma unroll
        for (int j = 0; j < N; j++)
            if (j < nb) {
                const float2 z = __ldg(j >= r ? M + r * nb + j : M + j * nb + r);
                hr[j] = z.x;
                hi[j] = j > r ? z.y : j < r ? -z.y : 0.0;
            }
    }
    for (int sweep = 0; sweep < P.sweeps; ++sweep) {
        double off = 0.0, all = 0.0;
#pragma unroll
        for (int j = 0; j < N; j++) {
            const double a2 = (r < nb) ? hr[j] * hr[j] + hi[j] * hi[j] : 0.0;
            all += a2;
            if (j != r) off += a2;
        }
#pragma unroll
        for (int d = 1; d < N; d <<= 1) {
            off += __shfl_xor_sync(mask, off, d);
            all += __shfl_xor_sync(mask, all, d);
        }
        if (!__any_sync(mask, live && off > 1e-24 * all)) break;
        JacobiSweep<N, 0>::run(hr, hi, vr, vi, r, base);
    }
    double lam[N];
#pragma unroll
    for (int c = 0; c < N; c++) lam[c] = __shfl_sync(mask, hr[c], base + c);
    if (!live) return;
#pragma unroll
    for (int c = 0; c < N; c++) {
        int rank = 0;
#pragma unroll
        for (int d = 0; d < N; d++) rank += (lam[d] < lam[c] || (lam[d] == lam[c] && d < c)) ? 1 : 0;
        if (rank < nb && r < nb) {
            if (r == 0) P.E[mat * nb + rank] = (float)lam[c];
            P.A[(mat * nb + rank) * nb + r] = make_float2((float)vr[c], (float)vi[c]);
        }
    }
}

}  // namespace tdos
