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
//    Joseph form stays at 0.09 x.
//  * Frames: C^s_n is carried in the frame the filtered state of layer n was stored in (momentum axes aimed at
//    the filtered momentum p^+_n); N comes out in the frame aimed at the propagated momentum p^-_n.  One
//    reaim_momentum call takes C^s_n from the first to the second.
#pragma once
#include "kf_math.cuh"

namespace kf {

// Symmetric 5 x 5 over (t, z, b1, b2, c) held as a full array (both triangles name the same values).
// Written on the number type F like the filter (kf_math.cuh); the library instantiates F = float only (the packed
// two-tracks-per-thread form, F = f2, gave identical results but ran slower: see kf_smooth.cu).
template <class F>
struct Sym5T {
    F m[5][5];
};
using Sym5 = Sym5T<float>;
using Sym5x2 = Sym5T<f2>;

template <class F>
__device__ __forceinline__ void sym5_from_track(const TrackT<F>& t, Sym5T<F>& P) {
    P.m[0][0] = t.c11; P.m[0][1] = P.m[1][0] = t.c12; P.m[0][2] = P.m[2][0] = t.c13;
    P.m[0][3] = P.m[3][0] = t.c14; P.m[0][4] = P.m[4][0] = t.c15;
    P.m[1][1] = t.c22; P.m[1][2] = P.m[2][1] = t.c23; P.m[1][3] = P.m[3][1] = t.c24; P.m[1][4] = P.m[4][1] = t.c25;
    P.m[2][2] = t.c33; P.m[2][3] = P.m[3][2] = t.c34; P.m[2][4] = P.m[4][2] = t.c35;
    P.m[3][3] = t.c44; P.m[3][4] = P.m[4][3] = t.c45;
    P.m[4][4] = t.c55;
}

template <class F>
__device__ __forceinline__ void track_from_sym5(const Sym5T<F>& P, TrackT<F>& t) {
    t.c00 = F(0.0f); t.c01 = F(0.0f); t.c02 = F(0.0f); t.c03 = F(0.0f); t.c04 = F(0.0f); t.c05 = F(0.0f);
    t.c11 = P.m[0][0]; t.c12 = P.m[0][1]; t.c13 = P.m[0][2]; t.c14 = P.m[0][3]; t.c15 = P.m[0][4];
    t.c22 = P.m[1][1]; t.c23 = P.m[1][2]; t.c24 = P.m[1][3]; t.c25 = P.m[1][4];
    t.c33 = P.m[2][2]; t.c34 = P.m[2][3]; t.c35 = P.m[2][4];
    t.c44 = P.m[3][3]; t.c45 = P.m[3][4];
    t.c55 = P.m[4][4];
}

// The smoothed state of the layer further out, as the recursion carries it.
template <class F>
struct SmoothedNextT {
    F x, y, z, px, py, pz;   // x^s_n (global coordinates)
    F fpx, fpy, fpz;         // p^+_n: the filtered momentum of layer n = the aim of the frame Cs is held in
    F fax, fay;              // position frame Cs is held in (rts_step_surface only; the barrel step does not need it)
    Sym5T<F> Cs;             // C^s_n in the frame layer n was stored in
};
using SmoothedNext = SmoothedNextT<float>;

template <class F>
struct SmoothedStateT {
    F x, y, z, px, py, pz;
};

// One backward step: t = filtered state of layer k in its local frame (radial row zero), Ln = constants of the
// next used layer n, nx = smoothed state of n.  On success returns 0, x^s_k in `s` and C^s_k in Cs_out (frame of
// t).  On failure (the crossing cannot be recomputed, N not positive definite, a non-finite result) returns the
// status bit(s) and writes nothing.  Pair form: both tracks take the step or neither does.
template <class F, bool ELOSS = false>
__device__ __forceinline__ typename num_traits<F>::status
rts_step(const TrackT<F>& t, arg<F> k, arg<F> ik, const LayerConst& Ln, int model, float mass2, const Bethe& el,
         const SmoothedNextT<F>& nx, SmoothedStateT<F>& s, Sym5T<F>& Cs_out) {
    using M_ = typename num_traits<F>::mask;
    CrossingT<F> o;
    const M_ reached = helix_to_radius(t, k, ik, Ln, o);
    if (!all_of(reached)) return select_u(reached, 0u, ST_PROP_FAIL);
    const F ms = ms_at_crossing(Ln, model, o, t.pz);
    // local Jacobian rows over (a2, z, b1, b2, c) of layer k  (kf_math.cuh: row t', row z', row b2')
    const F t1 = o.t1, t3 = o.t3, t4 = o.t4;
    const F z1 = o.z1, z3 = o.z3, z4 = o.z4, thk = o.thk;
    const F h1 = o.mu * o.g1, h3 = o.mu * o.g3, h4 = o.mu * o.g4;   // row b2' = e_b2 + (h1, 0, h3, h4, 0)
    Sym5T<F> P;
    sym5_from_track(t, P);
    // M = P F~^T (5 x 5)
    F M[5][5];
#pragma unroll
    for (int i = 0; i < 5; ++i) {
        M[i][0] = P.m[i][0] * t1 + P.m[i][2] * t3 + P.m[i][3] * t4;
        M[i][1] = P.m[i][1] + P.m[i][0] * z1 + P.m[i][2] * z3 + P.m[i][3] * z4 + P.m[i][4] * thk;
        M[i][2] = P.m[i][2];
        M[i][3] = P.m[i][3] + (P.m[i][0] * h1 + P.m[i][2] * h3 + P.m[i][3] * h4);
        M[i][4] = P.m[i][4];
    }
    // Highland process noise Q~ of layer n at the propagated momentum (same expression as transport_cov)
    const F pz = t.pz;
    const F p2 = o.pt2 + pz * pz;
    const F ip2 = rcp_fast(p2);
    const F th2 = ms * (p2 + mass2) * ip2 * ip2;
    const F qc = th2 * p2 * o.ipt;
    const F q22 = th2 * pz * pz, q24 = -(qc * pz), q33 = th2 * p2, q44 = qc * (p2 * o.ipt);
    // N = F~ M + Q~
    F N[5][5];
#pragma unroll
    for (int b = 0; b < 5; ++b) {
        N[0][b] = t1 * M[0][b] + t3 * M[2][b] + t4 * M[3][b];
        N[1][b] = M[1][b] + z1 * M[0][b] + z3 * M[2][b] + z4 * M[3][b] + thk * M[4][b];
        N[2][b] = M[2][b];
        N[3][b] = M[3][b] + (h1 * M[0][b] + h3 * M[2][b] + h4 * M[3][b]);
        N[4][b] = M[4][b];
    }
    N[2][2] += q22; N[2][4] += q24; N[4][2] += q24; N[3][3] += q33; N[4][4] += q44;
    // Process noise of the whole map k -> n as the recursion needs it again below (Joseph form): Q~, or J Q~ J^T
    // with the energy loss of reading A21
    F y22 = q22, y24 = q24, y33 = q33, y44 = q44;
    F lf(1.0f), lg(1.0f), lh(0.0f);          // J = [[g, 0, h], [0, f, 0], [0, 0, f]] on (b1, b2, c); identity without the option
    if constexpr (ELOSS && std::is_same<F, float>::value) {   // (compiled out of the kernel for geometries without the option)
        if (model & MODEL_ENERGY_LOSS) {
            // Reading A21: on arrival, after C' = F~ P F~^T + Q~, the momentum is scaled by f (direction kept) and the
            // covariance goes through J.  The map k -> n is then J F~: M -> M J^T, N -> J N J^T, Q~ -> J Q~ J^T.
            Eloss e;
            if (!energy_loss_factors(el, Ln, model, mass2, o.erx * o.elx + o.ery * o.ely, o.pt2, o.ipt, pz, false, e))
                return ST_PROP_FAIL;
            lf = e.f; lg = e.g; lh = e.h;
#pragma unroll
            for (int i = 0; i < 5; ++i) {      // columns (b1, b2, c) of M and of N
                M[i][2] = lg * M[i][2] + lh * M[i][4]; M[i][3] = lf * M[i][3]; M[i][4] = lf * M[i][4];
                N[i][2] = lg * N[i][2] + lh * N[i][4]; N[i][3] = lf * N[i][3]; N[i][4] = lf * N[i][4];
            }
#pragma unroll
            for (int b = 0; b < 5; ++b) {      // rows of N
                N[2][b] = lg * N[2][b] + lh * N[4][b]; N[3][b] = lf * N[3][b]; N[4][b] = lf * N[4][b];
            }
            const float a0 = lg * q22 + lh * q24, a2 = lg * q24 + lh * q44;     // row b1 of J Q~
            y22 = lg * a0 + lh * a2;
            y24 = lf * a2;
            y33 = lf * lf * q33;
            y44 = lf * lf * q44;
        }
    }
    // N = L D L^T (unit lower L), from the upper triangle
    F Lm[5][5], d[5], id[5];
    M_ pd = reached;
#pragma unroll
    for (int j = 0; j < 5; ++j) {
        F dj = N[j][j];
#pragma unroll
        for (int r = 0; r < j; ++r) dj -= (Lm[j][r] * Lm[j][r]) * d[r];
        d[j] = dj;
        pd = pd & (dj > 0.0f);
        id[j] = rcp_fast(dj);
#pragma unroll
        for (int i = j + 1; i < 5; ++i) {
            F v = N[j][i];
#pragma unroll
            for (int r = 0; r < j; ++r) v -= (Lm[i][r] * Lm[j][r]) * d[r];
            Lm[i][j] = v * id[j];
        }
    }
    if (!all_of(pd)) return select_u(pd, 0u, ST_S_NOT_PD);
    // A = M N^-1, row by row:  L y = m,  z = y / d,  L^T a = z
    F A[5][5];
#pragma unroll
    for (int i = 0; i < 5; ++i) {
        F y[5];
#pragma unroll
        for (int j = 0; j < 5; ++j) {
            F v = M[i][j];
#pragma unroll
            for (int r = 0; r < j; ++r) v -= Lm[j][r] * y[r];
            y[j] = v;
        }
#pragma unroll
        for (int j = 4; j >= 0; --j) {
            F v = y[j] * id[j];
#pragma unroll
            for (int r = j + 1; r < 5; ++r) v -= Lm[r][j] * A[i][r];
            A[i][j] = v;
        }
    }
    // x^s_n - x^-_n in the arrival frame of n (radial component dropped: second order, null direction of N)
    const F dx = nx.x - o.xn, dy = nx.y - o.yn;
    const F dpx = nx.px - lf * o.pxn, dpy = nx.py - lf * o.pyn;
    F D[5];
    D[0] = o.erx * dy - o.ery * dx;
    D[1] = nx.z - o.zn;
    D[2] = o.elx * dpx + o.ely * dpy;
    D[3] = o.elx * dpy - o.ely * dpx;
    D[4] = (nx.pz - lf * pz) - o.T * D[2];
    F dl[5];
#pragma unroll
    for (int i = 0; i < 5; ++i) dl[i] = A[i][0] * D[0] + A[i][1] * D[1] + A[i][2] * D[2] + A[i][3] * D[3] + A[i][4] * D[4];
    // C^s_n from the frame aimed at p^+_n to the frame aimed at p^-_n
    TrackT<F> w;
    track_from_sym5(nx.Cs, w);
    {
        const F ipf = rsqrt_fast(nx.fpx * nx.fpx + nx.fpy * nx.fpy);
        const F fx = nx.fpx * ipf, fy = nx.fpy * ipf;
        reaim_momentum<true>(w, o.elx * fx + o.ely * fy, o.elx * fy - o.ely * fx, nx.fpz * ipf, o.T);
    }
    Sym5T<F> Y;
    sym5_from_track(w, Y);
    Y.m[2][2] += y22; Y.m[2][4] += y24; Y.m[4][2] += y24; Y.m[3][3] += y33; Y.m[4][4] += y44;
    // B = I - A (J F~) = I - (A J) F~
    F B[5][5];
#pragma unroll
    for (int i = 0; i < 5; ++i) {
        const F a0 = A[i][0], a1 = A[i][1];
        const F a2 = A[i][2] * lg, a3 = A[i][3] * lf, a4 = A[i][2] * lh + A[i][4] * lf;    // row i of A J
        B[i][0] = -(a0 * t1 + a1 * z1 + a3 * h1);
        B[i][1] = -a1;
        B[i][2] = -(a0 * t3 + a1 * z3 + a2 + a3 * h3);
        B[i][3] = -(a0 * t4 + a1 * z4 + a3 + a3 * h4);
        B[i][4] = -(a1 * thk + a4);
        B[i][i] += 1.0f;
    }
    // C^s_k = B P B^T + A Y A^T (upper triangle)
    F probe(0.0f);
    Sym5T<F> C;
#pragma unroll
    for (int i = 0; i < 5; ++i) {
        F u[5], v[5];
#pragma unroll
        for (int j = 0; j < 5; ++j) {
            u[j] = B[i][0] * P.m[0][j] + B[i][1] * P.m[1][j] + B[i][2] * P.m[2][j] + B[i][3] * P.m[3][j] + B[i][4] * P.m[4][j];
            v[j] = A[i][0] * Y.m[0][j] + A[i][1] * Y.m[1][j] + A[i][2] * Y.m[2][j] + A[i][3] * Y.m[3][j] + A[i][4] * Y.m[4][j];
        }
#pragma unroll
        for (int j = i; j < 5; ++j) {
            const F c = (u[0] * B[j][0] + u[1] * B[j][1] + u[2] * B[j][2] + u[3] * B[j][3] + u[4] * B[j][4]) +
                        (v[0] * A[j][0] + v[1] * A[j][1] + v[2] * A[j][2] + v[3] * A[j][3] + v[4] * A[j][4]);
            C.m[i][j] = c;
            C.m[j][i] = c;
            probe += c * 0.0f;
        }
    }
    probe += (dl[0] + dl[1] + dl[2] + dl[3] + dl[4]) * 0.0f;
    const M_ fin = abs_(probe) < __int_as_float(0x7f800000);
    if (!all_of(fin)) return select_u(fin, 0u, ST_NONFINITE);
    // x^s_k = x^+_k + A (...) in the frame of layer k
    const F iptk = rsqrt_fast(t.px * t.px + t.py * t.py);
    const F lx = t.px * iptk, ly = t.py * iptk, Tk = t.pz * iptk;
    s.x = t.x - t.eay * dl[0];
    s.y = t.y + t.eax * dl[0];
    s.z = t.z + dl[1];
    s.px = t.px + lx * dl[2] - ly * dl[3];
    s.py = t.py + ly * dl[2] + lx * dl[3];
    s.pz = t.pz + dl[4] + Tk * dl[2];
    Cs_out = C;
    return select_u(fin, 0u, 0u);
}

// ---- the same step for geometries with endcap discs (reading A23) ---------------------------------------------
// A state that stands on a DISC has no variance along z instead of along the radius, so its five live coordinates
// are (r, t | b1, b2, c) instead of (t, z | b1, b2, c).  `type` 0 = barrel, 1 = disc; the 5 x 5 matrices below are
// over the live coordinates of the layer they belong to, in the order of the track's covariance fields
// (barrel: indices 1 2 3 4 5, disc: 0 1 3 4 5 of (a1, a2, z, b1, b2, c)).
__device__ __forceinline__ void sym5_from_track_surface(const Track& t, int type, Sym5& P) {
    if (type == 0) { sym5_from_track(t, P); return; }
    P.m[0][0] = t.c00; P.m[0][1] = P.m[1][0] = t.c01; P.m[0][2] = P.m[2][0] = t.c03;
    P.m[0][3] = P.m[3][0] = t.c04; P.m[0][4] = P.m[4][0] = t.c05;
    P.m[1][1] = t.c11; P.m[1][2] = P.m[2][1] = t.c13; P.m[1][3] = P.m[3][1] = t.c14; P.m[1][4] = P.m[4][1] = t.c15;
    P.m[2][2] = t.c33; P.m[2][3] = P.m[3][2] = t.c34; P.m[2][4] = P.m[4][2] = t.c35;
    P.m[3][3] = t.c44; P.m[3][4] = P.m[4][3] = t.c45;
    P.m[4][4] = t.c55;
}

__device__ __forceinline__ void track_from_sym5_surface(const Sym5& P, int type, Track& t) {
    if (type == 0) { track_from_sym5(P, t); return; }
    t.c02 = 0.0f; t.c12 = 0.0f; t.c22 = 0.0f; t.c23 = 0.0f; t.c24 = 0.0f; t.c25 = 0.0f;
    t.c00 = P.m[0][0]; t.c01 = P.m[0][1]; t.c03 = P.m[0][2]; t.c04 = P.m[0][3]; t.c05 = P.m[0][4];
    t.c11 = P.m[1][1]; t.c13 = P.m[1][2]; t.c14 = P.m[1][3]; t.c15 = P.m[1][4];
    t.c33 = P.m[2][2]; t.c34 = P.m[2][3]; t.c35 = P.m[2][4];
    t.c44 = P.m[3][3]; t.c45 = P.m[3][4];
    t.c55 = P.m[4][4];
}

// One backward step between surfaces of either kind: t = filtered state of layer k (position, momentum, position
// frame), P = its covariance over k's live coordinates, src = type of k, Ln = the next used layer n (a barrel only
// after a barrel: layers are met in list order, reading A23).  Same recursion and Joseph form as rts_step; the
// Jacobian is taken dense (5 x 5: rows r'/t' or t'/z', b1', b2', c' over k's live coordinates), and C^s_n is brought
// from the frames it was stored in (position frame of x^+_n, momentum aimed at p^+_n) to the arrival frames in both
// blocks -- on a disc both in-plane position coordinates are live, so the rotation between the two position frames
// is first order there.  Returns 0 or the status bits; writes nothing on failure.
template <bool ELOSS>
__device__ __forceinline__ uint32_t rts_step_surface(const Track& t, const Sym5& P, int src, float k, float ik,
                                                     const LayerConst& Ln, int model, float mass2, const Bethe& el,
                                                     const SmoothedNext& nx, SmoothedStateT<float>& s, Sym5& Cs_out) {
    const int dst = Ln.type;
    float Fs[5][5];
#pragma unroll
    for (int a = 0; a < 5; ++a)
#pragma unroll
        for (int b = 0; b < 5; ++b) Fs[a][b] = a == b && a >= 2 ? 1.0f : 0.0f;
    float xn, yn, wn, pxn, pyn, erx, ery, elx, ely, T, pt2, ipt, ms, cos_a;
    if (dst == 0) {
        if (src != 0) return ST_PROP_FAIL;
        Crossing o;
        if (!helix_to_radius(t, k, ik, Ln, o)) return ST_PROP_FAIL;
        ms = ms_at_crossing(Ln, model, o, t.pz);
        Fs[0][0] = o.t1; Fs[0][2] = o.t3; Fs[0][3] = o.t4;
        Fs[1][0] = o.z1; Fs[1][1] = 1.0f; Fs[1][2] = o.z3; Fs[1][3] = o.z4; Fs[1][4] = o.thk;
        Fs[3][0] = o.mu * o.g1; Fs[3][2] = o.mu * o.g3; Fs[3][3] = 1.0f + o.mu * o.g4;
        xn = o.xn; yn = o.yn; wn = o.zn; pxn = o.pxn; pyn = o.pyn; erx = o.erx; ery = o.ery; elx = o.elx; ely = o.ely;
        T = o.T; pt2 = o.pt2; ipt = o.ipt;
        cos_a = o.erx * o.elx + o.ery * o.ely;
    } else {
        DiscCrossing o;
        const uint32_t rc = helix_to_plane(t, k, ik, Ln, o);
        if (rc) return rc;
        ms = ms_at_disc(Ln, model, o, t.pz);
        // rows r', t' over (a1, a2, z, b1, b2, c) as in transport_cov_disc; row b2' = e_b2 + (0, 0, b2z, b2b, 0, b2c)
        const float R[6] = {o.pc, -o.ps, -o.ca * o.iT, o.nr - o.ca * o.thk, -o.nt, -o.ca * o.thk * o.iT};
        const float Tt[6] = {o.ps, o.pc, -o.sa * o.iT, o.nt - o.sa * o.thk, o.nr, -o.sa * o.thk * o.iT};
        const float b2z = k * o.iT, b2b = o.theta, b2c = o.theta * o.iT;
        const bool sb = src == 0;                                         // k's two live position coordinates: (a2, z) or (a1, a2)
        Fs[0][0] = sb ? R[1] : R[0]; Fs[0][1] = sb ? R[2] : R[1]; Fs[0][2] = R[3]; Fs[0][3] = R[4]; Fs[0][4] = R[5];
        Fs[1][0] = sb ? Tt[1] : Tt[0]; Fs[1][1] = sb ? Tt[2] : Tt[1]; Fs[1][2] = Tt[3]; Fs[1][3] = Tt[4]; Fs[1][4] = Tt[5];
        Fs[3][1] = src == 0 ? b2z : 0.0f; Fs[3][2] = b2b; Fs[3][3] = 1.0f; Fs[3][4] = b2c;
        xn = o.xn; yn = o.yn; wn = o.zt; pxn = o.pxn; pyn = o.pyn; erx = o.erx; ery = o.ery; elx = o.elx; ely = o.ely;
        T = o.T; pt2 = o.pt2; ipt = o.ipt;
        cos_a = o.T;                           // (path factor at a disc: |p| / |pz|, see fit_layer_disc)
    }
    // M = P Fs^T,  N = Fs M + Q~
    float M[5][5], N[5][5];
#pragma unroll
    for (int i = 0; i < 5; ++i)
#pragma unroll
        for (int j = 0; j < 5; ++j)
            M[i][j] = P.m[i][0] * Fs[j][0] + P.m[i][1] * Fs[j][1] + P.m[i][2] * Fs[j][2] + P.m[i][3] * Fs[j][3] + P.m[i][4] * Fs[j][4];
#pragma unroll
    for (int a = 0; a < 5; ++a)
#pragma unroll
        for (int b = 0; b < 5; ++b)
            N[a][b] = Fs[a][0] * M[0][b] + Fs[a][1] * M[1][b] + Fs[a][2] * M[2][b] + Fs[a][3] * M[3][b] + Fs[a][4] * M[4][b];
    const float pz = t.pz;
    const float p2 = pt2 + pz * pz;
    const float ip2 = rcp_fast(p2);
    const float th2 = ms * (p2 + mass2) * ip2 * ip2;
    const float qc = th2 * p2 * ipt;
    const float q22 = th2 * pz * pz, q24 = -(qc * pz), q33 = th2 * p2, q44 = qc * (p2 * ipt);
    N[2][2] += q22; N[2][4] += q24; N[4][2] += q24; N[3][3] += q33; N[4][4] += q44;
    float y22 = q22, y24 = q24, y33 = q33, y44 = q44;
    float lf = 1.0f, lg = 1.0f, lh = 0.0f;
    if constexpr (ELOSS) {
        if (model & MODEL_ENERGY_LOSS) {       // reading A21, as in rts_step: the map k -> n is J Fs
            Eloss e;
            if (!energy_loss_factors(el, Ln, model, mass2, cos_a, pt2, ipt, pz, false, e)) return ST_PROP_FAIL;
            lf = e.f; lg = e.g; lh = e.h;
#pragma unroll
            for (int i = 0; i < 5; ++i) {
                M[i][2] = lg * M[i][2] + lh * M[i][4]; M[i][3] = lf * M[i][3]; M[i][4] = lf * M[i][4];
                N[i][2] = lg * N[i][2] + lh * N[i][4]; N[i][3] = lf * N[i][3]; N[i][4] = lf * N[i][4];
            }
#pragma unroll
            for (int b = 0; b < 5; ++b) {
                N[2][b] = lg * N[2][b] + lh * N[4][b]; N[3][b] = lf * N[3][b]; N[4][b] = lf * N[4][b];
            }
            const float a0 = lg * q22 + lh * q24, a2 = lg * q24 + lh * q44;
            y22 = lg * a0 + lh * a2;
            y24 = lf * a2;
            y33 = lf * lf * q33;
            y44 = lf * lf * q44;
        }
    }
    // N = L D L^T,  A = M N^-1
    float Lm[5][5], d[5], id[5];
    bool pd = true;
#pragma unroll
    for (int j = 0; j < 5; ++j) {
        float dj = N[j][j];
#pragma unroll
        for (int r = 0; r < j; ++r) dj -= (Lm[j][r] * Lm[j][r]) * d[r];
        d[j] = dj;
        pd = pd && (dj > 0.0f);
        id[j] = rcp_fast(dj);
#pragma unroll
        for (int i = j + 1; i < 5; ++i) {
            float v = N[j][i];
#pragma unroll
            for (int r = 0; r < j; ++r) v -= (Lm[i][r] * Lm[j][r]) * d[r];
            Lm[i][j] = v * id[j];
        }
    }
    if (!pd) return ST_S_NOT_PD;
    float A[5][5];
#pragma unroll
    for (int i = 0; i < 5; ++i) {
        float y[5];
#pragma unroll
        for (int j = 0; j < 5; ++j) {
            float v = M[i][j];
#pragma unroll
            for (int r = 0; r < j; ++r) v -= Lm[j][r] * y[r];
            y[j] = v;
        }
#pragma unroll
        for (int j = 4; j >= 0; --j) {
            float v = y[j] * id[j];
#pragma unroll
            for (int r = j + 1; r < 5; ++r) v -= Lm[r][j] * A[i][r];
            A[i][j] = v;
        }
    }
    // x^s_n - x^-_n over n's live coordinates, in the arrival frames
    const float dx = nx.x - xn, dy = nx.y - yn;
    const float dpx = nx.px - lf * pxn, dpy = nx.py - lf * pyn;
    float D[5];
    const float dr = erx * dx + ery * dy, dt = erx * dy - ery * dx;
    D[0] = dst == 0 ? dt : dr;
    D[1] = dst == 0 ? nx.z - wn : dt;
    D[2] = elx * dpx + ely * dpy;
    D[3] = elx * dpy - ely * dpx;
    D[4] = (nx.pz - lf * pz) - T * D[2];
    float dl[5];
#pragma unroll
    for (int i = 0; i < 5; ++i) dl[i] = A[i][0] * D[0] + A[i][1] * D[1] + A[i][2] * D[2] + A[i][3] * D[3] + A[i][4] * D[4];
    // C^s_n: stored frames -> arrival frames (position block, then momentum block)
    Track w;
    track_from_sym5_surface(nx.Cs, dst, w);
    if (dst == 0) { w.c00 = 0.0f; w.c01 = 0.0f; w.c02 = 0.0f; w.c03 = 0.0f; w.c04 = 0.0f; w.c05 = 0.0f; }
    reframe_position(w, erx * nx.fax + ery * nx.fay, erx * nx.fay - ery * nx.fax);
    {
        const float ipf = rsqrt_fast(nx.fpx * nx.fpx + nx.fpy * nx.fpy);
        const float fx = nx.fpx * ipf, fy = nx.fpy * ipf;
        reaim_momentum<false>(w, elx * fx + ely * fy, elx * fy - ely * fx, nx.fpz * ipf, T);
    }
    Sym5 Y;
    sym5_from_track_surface(w, dst, Y);
    Y.m[2][2] += y22; Y.m[2][4] += y24; Y.m[4][2] += y24; Y.m[3][3] += y33; Y.m[4][4] += y44;
    // B = I - (A J) Fs
    float B[5][5];
#pragma unroll
    for (int i = 0; i < 5; ++i) {
        const float a0 = A[i][0], a1 = A[i][1];
        const float a2 = A[i][2] * lg, a3 = A[i][3] * lf, a4 = A[i][2] * lh + A[i][4] * lf;
#pragma unroll
        for (int m = 0; m < 5; ++m)
            B[i][m] = (i == m ? 1.0f : 0.0f) - (a0 * Fs[0][m] + a1 * Fs[1][m] + a2 * Fs[2][m] + a3 * Fs[3][m] + a4 * Fs[4][m]);
    }
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
    // x^s_k = x^+_k + A (...) over k's live coordinates
    const float iptk = rsqrt_fast(t.px * t.px + t.py * t.py);
    const float lx = t.px * iptk, ly = t.py * iptk, Tk = t.pz * iptk;
    const float sr = src == 0 ? 0.0f : dl[0], st_ = src == 0 ? dl[0] : dl[1];
    s.x = t.x + t.eax * sr - t.eay * st_;
    s.y = t.y + t.eay * sr + t.eax * st_;
    s.z = src == 0 ? t.z + dl[1] : t.z;
    s.px = t.px + lx * dl[2] - ly * dl[3];
    s.py = t.py + ly * dl[2] + lx * dl[3];
    s.pz = t.pz + dl[4] + Tk * dl[2];
    Cs_out = C;
    return 0u;
}

// A 5 x 5 covariance held in the frame of track `f` (position frame (eax, eay), momentum axes aimed at f's
// momentum) -> the 21 packed elements in global coordinates, returned in g's covariance fields.
template <class F>
__device__ __forceinline__ void sym5_to_global(const Sym5T<F>& C, const TrackT<F>& f, TrackT<F>& g) {
    g = f;
    track_from_sym5(C, g);
    leave_local_frame(g);
}

}  // namespace kf
