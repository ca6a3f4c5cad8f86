// kf_rts.cuh -- one step of the fixed-interval (Rauch-Tung-Striebel) smoother in the kernels' track-local frame.
//
// PAPER.md:57 (section 2): the last stage of tracking is "a final fit with a KF and smoother".  DESIGN.md reading
// A22: the smoother is the RTS recursion over the layers the forward filter used, on the model that filter
// linearised.  With x^+_k, C^+_k the filtered state of layer k, x^-_n, C^-_n the prediction for the next used
// layer n and G the Jacobian of the map between them,
//     A     = C^+_k G^T (C^-_n)^+,   x^s_k = x^+_k + A (x^s_n - x^-_n),   C^s_k = C^+_k + A (C^s_n - C^-_n) A^T.
//
// HOW it is computed here (what differs from the textbook form and why):
//  * The forward kernel stores, per used layer, the filtered state in the LOCAL frame (6 state values, the 15
//    live covariance elements, the position frame).  The backward kernel recomputes the crossing k -> n from it
//    (helix_to_radius, same arithmetic as the filter), which gives x^-_n, the 5 x 5 local Jacobian F~ (identity
//    plus the rows tau, zeta and mu G_r of kf_math.cuh) and N = C^-_n = F~ P F~^T + Q~ without storing any of them.
//  * In the local frame every matrix is 5 x 5 over (t, z, b1, b2, c): the radial row of a covariance that was
//    transported to a cylinder is identically zero, so the pseudo-inverse of the textbook form is the plain
//    inverse of the 5 x 5 block (LDL^T, five reciprocals).
//  * The covariance uses the JOSEPH form of the same recursion,
//        C^s_k = (I - A F~) P (I - A F~)^T + A (C^s_n + Q~) A^T,
//    algebraically identical (P - A N A^T = (I - A F~) P (I - A F~)^T + A Q~ A^T because A N = P F~^T) but a
//    sum of positive semi-definite terms.  The textbook difference P + A (C^s_n - N) A^T cancels 3 - 4 digits on
//    the inner layers, where the filtered momentum variance is the 30 % prior and the smoothed one is the full
//    track's: measured in fp32 on config 3 it misses the 1e-3 covariance tolerance (1.7 x) at layer 0, the
//    Joseph form stays at 0.09 x (profiles/r02_smoother.md).
//  * Frames: C^s_n is carried in the frame the filtered state of layer n was stored in (momentum axes aimed at
//    the filtered momentum p^+_n); N comes out in the frame aimed at the propagated momentum p^-_n.  One
//    reaim_momentum call takes C^s_n from the first to the second.
#pragma once
#include "kf_math.cuh"

namespace kf {

// Symmetric 5 x 5 over (t, z, b1, b2, c) held as a full array (both triangles name the same values).
struct Sym5 {
    float m[5][5];
};

__device__ __forceinline__ void sym5_from_track(const Track& t, Sym5& P) {
    P.m[0][0] = t.c11; P.m[0][1] = P.m[1][0] = t.c12; P.m[0][2] = P.m[2][0] = t.c13;
    P.m[0][3] = P.m[3][0] = t.c14; P.m[0][4] = P.m[4][0] = t.c15;
    P.m[1][1] = t.c22; P.m[1][2] = P.m[2][1] = t.c23; P.m[1][3] = P.m[3][1] = t.c24; P.m[1][4] = P.m[4][1] = t.c25;
    P.m[2][2] = t.c33; P.m[2][3] = P.m[3][2] = t.c34; P.m[2][4] = P.m[4][2] = t.c35;
    P.m[3][3] = t.c44; P.m[3][4] = P.m[4][3] = t.c45;
    P.m[4][4] = t.c55;
}

__device__ __forceinline__ void track_from_sym5(const Sym5& P, Track& t) {
    t.c00 = 0.0f; t.c01 = 0.0f; t.c02 = 0.0f; t.c03 = 0.0f; t.c04 = 0.0f; t.c05 = 0.0f;
    t.c11 = P.m[0][0]; t.c12 = P.m[0][1]; t.c13 = P.m[0][2]; t.c14 = P.m[0][3]; t.c15 = P.m[0][4];
    t.c22 = P.m[1][1]; t.c23 = P.m[1][2]; t.c24 = P.m[1][3]; t.c25 = P.m[1][4];
    t.c33 = P.m[2][2]; t.c34 = P.m[2][3]; t.c35 = P.m[2][4];
    t.c44 = P.m[3][3]; t.c45 = P.m[3][4];
    t.c55 = P.m[4][4];
}

// The smoothed state of the layer further out, as the recursion carries it.
struct SmoothedNext {
    float x, y, z, px, py, pz;   // x^s_n (global coordinates)
    float fpx, fpy, fpz;         // p^+_n: the filtered momentum of layer n = the aim of the frame Cs is held in
    Sym5 Cs;                     // C^s_n in the frame layer n was stored in
};

// One backward step: t = filtered state of layer k in its local frame (radial row zero), Ln = constants of the
// next used layer n, nx = smoothed state of n.  On success returns 0, x^s_k in (sx, sy, sz, spx, spy, spz) and
// C^s_k in Cs_out (frame of t).  On failure (the crossing cannot be recomputed, N not positive definite, a
// non-finite result) returns the status bit and writes nothing.
__device__ __forceinline__ uint32_t rts_step(const Track& t, float k, float ik, const LayerConst& Ln, int model,
                                             float mass2, const SmoothedNext& nx, float& sx, float& sy, float& sz,
                                             float& spx, float& spy, float& spz, Sym5& Cs_out) {
    Crossing o;
    if (!helix_to_radius(t, k, ik, Ln, o)) return ST_PROP_FAIL;
    const float ms = ms_at_crossing(Ln, model, o, t.pz);
    // local Jacobian rows over (a2, z, b1, b2, c) of layer k  (kf_math.cuh: row t', row z', row b2')
    const float t1 = o.t1, t3 = o.t3, t4 = o.t4;
    const float z1 = o.z1, z3 = o.z3, z4 = o.z4, thk = o.thk;
    const float h1 = o.mu * o.g1, h3 = o.mu * o.g3, h4 = o.mu * o.g4;   // row b2' = e_b2 + (h1, 0, h3, h4, 0)
    Sym5 P;
    sym5_from_track(t, P);
    // M = P F~^T (5 x 5)
    float M[5][5];
#pragma unroll
    for (int i = 0; i < 5; ++i) {
        M[i][0] = P.m[i][0] * t1 + P.m[i][2] * t3 + P.m[i][3] * t4;
        M[i][1] = P.m[i][1] + P.m[i][0] * z1 + P.m[i][2] * z3 + P.m[i][3] * z4 + P.m[i][4] * thk;
        M[i][2] = P.m[i][2];
        M[i][3] = P.m[i][3] + (P.m[i][0] * h1 + P.m[i][2] * h3 + P.m[i][3] * h4);
        M[i][4] = P.m[i][4];
    }
    // Highland process noise Q~ of layer n at the propagated momentum (same expression as transport_cov)
    const float pz = t.pz;
    const float p2 = o.pt2 + pz * pz;
    const float ip2 = rcp_fast(p2);
    const float th2 = ms * (p2 + mass2) * ip2 * ip2;
    const float qc = th2 * p2 * o.ipt;
    const float q22 = th2 * pz * pz, q24 = -qc * pz, q33 = th2 * p2, q44 = qc * (p2 * o.ipt);
    // N = F~ M + Q~ (upper triangle, then mirrored)
    float N[5][5];
#pragma unroll
    for (int b = 0; b < 5; ++b) {
        N[0][b] = t1 * M[0][b] + t3 * M[2][b] + t4 * M[3][b];
        N[1][b] = M[1][b] + z1 * M[0][b] + z3 * M[2][b] + z4 * M[3][b] + thk * M[4][b];
        N[2][b] = M[2][b];
        N[3][b] = M[3][b] + (h1 * M[0][b] + h3 * M[2][b] + h4 * M[3][b]);
        N[4][b] = M[4][b];
    }
    N[2][2] += q22; N[2][4] += q24; N[4][2] += q24; N[3][3] += q33; N[4][4] += q44;
    // N = L D L^T (unit lower L), symmetrised from the upper triangle
    float Lm[5][5], d[5], id[5];
    bool pd = true;
#pragma unroll
    for (int j = 0; j < 5; ++j) {
        float dj = N[j][j];
#pragma unroll
        for (int s = 0; s < j; ++s) dj -= Lm[j][s] * Lm[j][s] * d[s];
        d[j] = dj;
        pd = pd && (dj > 0.0f);
        id[j] = rcp_fast(dj);
#pragma unroll
        for (int i = j + 1; i < 5; ++i) {
            float v = N[j][i];
#pragma unroll
            for (int s = 0; s < j; ++s) v -= Lm[i][s] * Lm[j][s] * d[s];
            Lm[i][j] = v * id[j];
        }
    }
    if (!pd) return ST_S_NOT_PD;
    // A = M N^-1, row by row:  L y = m,  z = y / d,  L^T a = z
    float A[5][5];
#pragma unroll
    for (int i = 0; i < 5; ++i) {
        float y[5];
#pragma unroll
        for (int j = 0; j < 5; ++j) {
            float v = M[i][j];
#pragma unroll
            for (int s = 0; s < j; ++s) v -= Lm[j][s] * y[s];
            y[j] = v;
        }
#pragma unroll
        for (int j = 4; j >= 0; --j) {
            float v = y[j] * id[j];
#pragma unroll
            for (int s = j + 1; s < 5; ++s) v -= Lm[s][j] * A[i][s];
            A[i][j] = v;
        }
    }
    // x^s_n - x^-_n in the arrival frame of n (radial component dropped: second order, null direction of N)
    const float dx = nx.x - o.xn, dy = nx.y - o.yn;
    const float dpx = nx.px - o.pxn, dpy = nx.py - o.pyn;
    float D[5];
    D[0] = o.erx * dy - o.ery * dx;
    D[1] = nx.z - o.zn;
    D[2] = o.elx * dpx + o.ely * dpy;
    D[3] = o.elx * dpy - o.ely * dpx;
    D[4] = (nx.pz - pz) - o.T * D[2];
    float dl[5];
#pragma unroll
    for (int i = 0; i < 5; ++i) dl[i] = A[i][0] * D[0] + A[i][1] * D[1] + A[i][2] * D[2] + A[i][3] * D[3] + A[i][4] * D[4];
    // C^s_n from the frame aimed at p^+_n to the frame aimed at p^-_n
    Track w;
    track_from_sym5(nx.Cs, w);
    {
        const float ipf = rsqrt_fast(nx.fpx * nx.fpx + nx.fpy * nx.fpy);
        const float fx = nx.fpx * ipf, fy = nx.fpy * ipf;
        reaim_momentum<true>(w, o.elx * fx + o.ely * fy, o.elx * fy - o.ely * fx, nx.fpz * ipf, o.T);
    }
    Sym5 Y;
    sym5_from_track(w, Y);
    Y.m[2][2] += q22; Y.m[2][4] += q24; Y.m[4][2] += q24; Y.m[3][3] += q33; Y.m[4][4] += q44;
    // B = I - A F~
    float B[5][5];
#pragma unroll
    for (int i = 0; i < 5; ++i) {
        B[i][0] = -(A[i][0] * t1 + A[i][1] * z1 + A[i][3] * h1);
        B[i][1] = -A[i][1];
        B[i][2] = -(A[i][0] * t3 + A[i][1] * z3 + A[i][2] + A[i][3] * h3);
        B[i][3] = -(A[i][0] * t4 + A[i][1] * z4 + A[i][3] + A[i][3] * h4);
        B[i][4] = -(A[i][1] * thk + A[i][4]);
        B[i][i] += 1.0f;
    }
    // C^s_k = B P B^T + A Y A^T (upper triangle)
    float probe = 0.0f;
    Sym5 C;
#pragma unroll
    for (int i = 0; i < 5; ++i) {
        float u[5], v[5];
#pragma unroll
        for (int j = 0; j < 5; ++j) {
            u[j] = B[i][0] * P.m[0][j] + B[i][1] * P.m[1][j] + B[i][2] * P.m[2][j] + B[i][3] * P.m[3][j] + B[i][4] * P.m[4][j];
            v[j] = A[i][0] * Y.m[0][j] + A[i][1] * Y.m[1][j] + A[i][2] * Y.m[2][j] + A[i][3] * Y.m[3][j] + A[i][4] * Y.m[4][j];
        }
#pragma unroll
        for (int j = i; j < 5; ++j) {
            const float c = (u[0] * B[j][0] + u[1] * B[j][1] + u[2] * B[j][2] + u[3] * B[j][3] + u[4] * B[j][4]) +
                            (v[0] * A[j][0] + v[1] * A[j][1] + v[2] * A[j][2] + v[3] * A[j][3] + v[4] * A[j][4]);
            C.m[i][j] = c;
            C.m[j][i] = c;
            probe += c * 0.0f;
        }
    }
    probe += (dl[0] + dl[1] + dl[2] + dl[3] + dl[4]) * 0.0f;
    if (!(fabsf(probe) < __int_as_float(0x7f800000))) return ST_NONFINITE;
    // x^s_k = x^+_k + A (...) in the frame of layer k
    const float iptk = rsqrt_fast(t.px * t.px + t.py * t.py);
    const float lx = t.px * iptk, ly = t.py * iptk, Tk = t.pz * iptk;
    sx = t.x - t.eay * dl[0];
    sy = t.y + t.eax * dl[0];
    sz = t.z + dl[1];
    spx = t.px + lx * dl[2] - ly * dl[3];
    spy = t.py + ly * dl[2] + lx * dl[3];
    spz = t.pz + dl[4] + Tk * dl[2];
    Cs_out = C;
    return 0u;
}

// A 5 x 5 covariance held in the frame of track `f` (position frame (eax, eay), momentum axes aimed at f's
// momentum) -> the 21 packed elements in global coordinates, returned in g's covariance fields.
__device__ __forceinline__ void sym5_to_global(const Sym5& C, const Track& f, Track& g) {
    g = f;
    track_from_sym5(C, g);
    leave_local_frame(g);
}

}  // namespace kf
