// lbm_node.cuh -- register-resident per-node arithmetic of the fused update: moments (eq. 1,
// P:85), Guo velocity shift (eq. 16), equilibrium (eq. 3), LBGK relaxation
// (Alg. 1 l.13), MRT relaxation (eq. 4) and Guo source (eq. 17).
//
// Everything works on the DEVIATION h_i = f_i - w_i from the rest equilibrium at rho = 1 (the
// round-off-minimising storage the paper recommends; reading A12).  The
// collision is affine in f, so it carries over unchanged: sum_i h_i = rho - 1, sum_i h_i e_i = j,
// h_i^eq = w_i (drho + rho (3 e.v + 4.5 (e.v)^2 - 1.5 v.v)).
#pragma once
#include <cmath>
#include "lbm_lattice.cuh"

namespace lbm {

// Parameters of one component's collision, passed to kernels by value (constant bank).
template <typename T> struct Relax {
    T inv_tau;        // omega = 1 / tau, rounded to T such that 1 - omega is also a T (set_bgk)
    T keep;           // 1 - omega, exactly
    T src_scale;      // 1 - omega / 2, prefactor of eq. (17)
    // omega / 36 and (1 - omega / 2) / 36 as unevaluated sums hi + lo of two T (see collide()):
    T om36_hi, om36_lo, sc36_hi, sc36_lo;
    T i36_hi, i36_lo; // 1 / 36 likewise (Exact Difference Method)
    T tau0, cs2x36;   // Smagorinsky: molecular tau_0 and 4 c_s^-4 C_S^2 = 36 C_S^2 of eq. (9)
    T in[19];         // MRT: 1 / |M_k|^2 (Exact Difference Method increment)
    T g[3];           // body acceleration
    T ubc[3];         // velocity imposed on equilibrium-velocity nodes (reading A21)
    T cr[19];         // MRT: rate_k / |M_k|^2                 (relaxation, eq. 4)
    T cs[19];         // MRT: (1 - rate_k / 2) / |M_k|^2       (source, reading A16)
};

// Fill the LBGK constants for relaxation time tau.  omega is rounded to T once and every other
// constant is derived from that rounded value, so that the collision conserves mass and momentum
// for the omega it actually uses.
template <typename T> inline void set_bgk(Relax<T> &r, double tau) {
    // pick the pair (omega, 1 - omega) so that both are representable: for omega in [1/2, 2] the
    // difference 1 - fl(omega) is exact (Sterbenz); below 1/2 round 1 - omega first and take
    // omega = 1 - fl(1 - omega), exact for the same reason.
    if (1.0 / tau >= 0.5) { r.inv_tau = T(1.0 / tau); r.keep = T(1) - r.inv_tau; }
    else { r.keep = T(1.0 - 1.0 / tau); r.inv_tau = T(1) - r.keep; }
    const double om = double(r.inv_tau), c = om / 36.0, s = (1.0 - 0.5 * om) / 36.0;
    r.src_scale = T(1.0 - 0.5 * om);
    r.om36_hi = T(c); r.om36_lo = T(c - double(r.om36_hi));
    r.sc36_hi = T(s); r.sc36_lo = T(s - double(r.sc36_hi));
    r.i36_hi = T(1.0 / 36.0); r.i36_lo = T(1.0 / 36.0 - double(r.i36_hi));
    r.tau0 = T(tau); r.cs2x36 = T(0);
}

template <class L, typename T> LBM_HD void moments(const T (&h)[L::Q], T &drho, T (&j)[3]) {
    T s = h[0], jx = T(0), jy = T(0), jz = T(0);
#pragma unroll
    for (int i = 1; i < L::Q; i++) {
        s += h[i];
        if (L::ex(i) == 1) jx += h[i]; else if (L::ex(i) == -1) jx -= h[i];
        if (L::ey(i) == 1) jy += h[i]; else if (L::ey(i) == -1) jy -= h[i];
        if (L::ez(i) == 1) jz += h[i]; else if (L::ez(i) == -1) jz -= h[i];
    }
    drho = s; j[0] = jx; j[1] = jy; j[2] = jz;
}

template <class L, typename T> LBM_HD T e_dot(int i, const T (&a)[3]) {
    T s = T(0);
    if (L::ex(i) == 1) s += a[0]; else if (L::ex(i) == -1) s -= a[0];
    if (L::ey(i) == 1) s += a[1]; else if (L::ey(i) == -1) s -= a[1];
    if (L::ez(i) == 1) s += a[2]; else if (L::ez(i) == -1) s -= a[2];
    return s;
}

// Second moments P_ab = sum_i e_ia e_ib h_i in the order xx, yy, zz, xy, yz, xz, and e_i.P.e_i.
template <class L, typename T> LBM_HD void second_moments(const T (&h)[L::Q], T (&P)[6]) {
#pragma unroll
    for (int c = 0; c < 6; c++) P[c] = T(0);
#pragma unroll
    for (int i = 1; i < L::Q; i++) {
        const int x = L::ex(i), y = L::ey(i), z = L::ez(i);
        if (x) P[0] += h[i];
        if (y) P[1] += h[i];
        if (z) P[2] += h[i];
        if (x * y == 1) P[3] += h[i]; else if (x * y == -1) P[3] -= h[i];
        if (y * z == 1) P[4] += h[i]; else if (y * z == -1) P[4] -= h[i];
        if (x * z == 1) P[5] += h[i]; else if (x * z == -1) P[5] -= h[i];
    }
}
template <class L, typename T> LBM_HD T e_quad(int i, const T (&P)[6]) {
    const int x = L::ex(i), y = L::ey(i), z = L::ez(i);
    T s = T(0);
    if (x) s += P[0];
    if (y) s += P[1];
    if (z) s += P[2];
    if (x * y == 1) s += T(2) * P[3]; else if (x * y == -1) s -= T(2) * P[3];
    if (y * z == 1) s += T(2) * P[4]; else if (y * z == -1) s -= T(2) * P[4];
    if (x * z == 1) s += T(2) * P[5]; else if (x * z == -1) s -= T(2) * P[5];
    return s;
}

// h_i^eq for all i, eq. (3) minus w_i.
template <class L, typename T>
LBM_HD void equilibrium_dev(T rho, T drho, const T (&v)[3], T (&heq)[L::Q]) {
    const T vv15 = T(1.5) * (v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
#pragma unroll
    for (int i = 0; i < L::Q; i++) {
        const T ev = e_dot<L, T>(i, v);
        heq[i] = L::template w<T>(i) * (drho + rho * (T(3) * ev + T(4.5) * ev * ev - vv15));
    }
}

// Bracket of eq. (17): w_i [3 (e_i - v) + 9 (e_i.v) e_i] . F
template <class L, typename T>
LBM_HD void guo_bracket(const T (&v)[3], const T (&F)[3], T (&src)[L::Q]) {
    const T vF = v[0] * F[0] + v[1] * F[1] + v[2] * F[2];
#pragma unroll
    for (int i = 0; i < L::Q; i++) {
        const T ev = e_dot<L, T>(i, v), eF = e_dot<L, T>(i, F);
        src[i] = L::template w<T>(i) * (T(3) * (eF - vF) + T(9) * ev * eF);
    }
}

// ---- MRT moment transforms (eq. 4; basis = reading A5) -------------------------------
// m = M d and o = M^T r.  Rows of M are mutually orthogonal polynomials of e_i with small
// integer entries; both transforms are hand-factored through the velocity-class sub-sums so the
// pair costs ~170 flop instead of the ~1400 of two dense 19x19 products (keeps MRT HBM-bound).
template <class L, typename T> struct Mrt;

template <typename T> struct Mrt<D3Q19, T> {
    static constexpr bool closed_form_meq = true;
    // M (f^eq - w) in closed form (reading A6: m^eq = M f^eq with eq. (3)); the coefficients are
    // sum_i M_ki w_i {1, 3 e_ia, 4.5 e_ia e_ib - 1.5 delta_ab}, which for this basis reduce to
    // d'Humieres' equilibrium moments with w_eps = 3, w_epsj = -11/2, w_xx = -1/2.
    LBM_HD static void meq_dev(T rho, T drho, const T (&v)[3], T (&q)[19]) {
        const T xx = v[0] * v[0], yy = v[1] * v[1], zz = v[2] * v[2];
        const T rvv = rho * (xx + yy + zz);
        const T jx = rho * v[0], jy = rho * v[1], jz = rho * v[2];
        q[0] = drho;
        q[1] = T(19) * rvv - T(11) * drho;
        q[2] = T(3) * drho - T(5.5) * rvv;
        q[3] = jx; q[4] = T(-2.0 / 3.0) * jx;
        q[5] = jy; q[6] = T(-2.0 / 3.0) * jy;
        q[7] = jz; q[8] = T(-2.0 / 3.0) * jz;
        q[9] = rho * (T(2) * xx - yy - zz); q[10] = T(-0.5) * q[9];
        q[11] = rho * (yy - zz);            q[12] = T(-0.5) * q[11];
        q[13] = jx * v[1]; q[14] = jy * v[2]; q[15] = jx * v[2];
        q[16] = T(0); q[17] = T(0); q[18] = T(0);
    }
    static constexpr double norm(int k) {
        constexpr double n[19] = {19, 2394, 252, 10, 40, 10, 40, 10, 40, 36, 72, 12, 24, 4, 4, 4, 8, 8, 8};
        return n[k];
    }
    LBM_HD static void forward(const T (&d)[19], T (&m)[19]) {
        const T Sx = d[1] + d[2], Dx = d[1] - d[2];
        const T Sy = d[3] + d[4], Dy = d[3] - d[4];
        const T Sz = d[5] + d[6], Dz = d[5] - d[6];
        // xy diagonals 7 (+,+) 8 (-,+) 9 (+,-) 10 (-,-)
        const T a1 = d[7] + d[10], a2 = d[8] + d[9], a3 = d[7] - d[10], a4 = d[9] - d[8];
        const T Sxy = a1 + a2, Pxy = a1 - a2, Xxy = a3 + a4, Yxy = a3 - a4;
        // xz diagonals 11 (+,+) 12 (-,+) 13 (+,-) 14 (-,-)
        const T b1 = d[11] + d[14], b2 = d[12] + d[13], b3 = d[11] - d[14], b4 = d[13] - d[12];
        const T Sxz = b1 + b2, Pxz = b1 - b2, Xxz = b3 + b4, Zxz = b3 - b4;
        // yz diagonals 15 (+,+) 16 (-,+) 17 (+,-) 18 (-,-)
        const T c1 = d[15] + d[18], c2 = d[16] + d[17], c3 = d[15] - d[18], c4 = d[17] - d[16];
        const T Syz = c1 + c2, Pyz = c1 - c2, Yyz = c3 + c4, Zyz = c3 - c4;
        const T A = Sx + Sy + Sz, B = Sxy + Sxz + Syz;
        const T Xd = Xxy + Xxz, Yd = Yxy + Yyz, Zd = Zxz + Zyz;
        const T axx = T(2) * Sx - Sy - Sz, dxx = Sxy + Sxz - T(2) * Syz;
        const T aww = Sy - Sz, dww = Sxy - Sxz;
        m[0] = d[0] + A + B;
        m[1] = T(-30) * d[0] - T(11) * A + T(8) * B;
        m[2] = T(12) * d[0] - T(4) * A + B;
        m[3] = Dx + Xd;  m[4] = Xd - T(4) * Dx;
        m[5] = Dy + Yd;  m[6] = Yd - T(4) * Dy;
        m[7] = Dz + Zd;  m[8] = Zd - T(4) * Dz;
        m[9] = axx + dxx;   m[10] = dxx - T(2) * axx;
        m[11] = aww + dww;  m[12] = dww - T(2) * aww;
        m[13] = Pxy; m[14] = Pyz; m[15] = Pxz;
        m[16] = Xxy - Xxz; m[17] = Yyz - Yxy; m[18] = Zxz - Zyz;
    }
    // o_i = sum_k M[k][i] r_k
    LBM_HD static void backward(const T (&r)[19], T (&o)[19]) {
        const T ca = r[0] - T(11) * r[1] - T(4) * r[2];   // axis class
        const T cd = r[0] + T(8) * r[1] + r[2];           // diagonal class
        o[0] = r[0] - T(30) * r[1] + T(12) * r[2];
        const T ax = ca + T(2) * (r[9] - T(2) * r[10]), lx = r[3] - T(4) * r[4];
        const T t1 = T(2) * r[10] - r[9], t2 = r[11] - T(2) * r[12];
        const T ay = ca + t1 + t2, ly = r[5] - T(4) * r[6];
        const T az = ca + t1 - t2, lz = r[7] - T(4) * r[8];
        o[1] = ax + lx; o[2] = ax - lx;
        o[3] = ay + ly; o[4] = ay - ly;
        o[5] = az + lz; o[6] = az - lz;
        const T qx = r[3] + r[4], qy = r[5] + r[6], qz = r[7] + r[8];
        const T s9 = r[9] + r[10], s11 = r[11] + r[12];
        {   // xy: cd + sx(qx + r16) + sy(qy - r17) + s9 + s11 + sx sy r13
            const T base = cd + s9 + s11, X = qx + r[16], Y = qy - r[17];
            const T p = base + r[13], q = base - r[13];
            o[7] = p + X + Y; o[10] = p - X - Y; o[8] = q - X + Y; o[9] = q + X - Y;
        }
        {   // xz: cd + sx(qx - r16) + sz(qz + r18) + s9 - s11 + sx sz r15
            const T base = cd + s9 - s11, X = qx - r[16], Z = qz + r[18];
            const T p = base + r[15], q = base - r[15];
            o[11] = p + X + Z; o[14] = p - X - Z; o[12] = q - X + Z; o[13] = q + X - Z;
        }
        {   // yz: cd + sy(qy + r17) + sz(qz - r18) - 2 s9 + sy sz r14
            const T base = cd - T(2) * s9, Y = qy + r[17], Z = qz - r[18];
            const T p = base + r[14], q = base - r[14];
            o[15] = p + Y + Z; o[18] = p - Y - Z; o[16] = q - Y + Z; o[17] = q + Y - Z;
        }
    }
};

// D2Q9 (reading A5): rows 1; -4+3n^2; 4-21n^2/2+9n^4/2; ex; (-5+3n^2)ex; ey; (-5+3n^2)ey;
// ex^2-ey^2; ex ey.  9x9 is small enough to unroll as constants.
template <typename T> struct Mrt<D2Q9, T> {
    static constexpr bool closed_form_meq = false;  // not in the configs: m^eq through M f^eq
    LBM_HD static void meq_dev(T, T, const T (&)[3], T (&)[9]) {}
    static constexpr double norm(int k) {
        constexpr double n[9] = {9, 36, 36, 6, 12, 6, 12, 4, 4};
        return n[k];
    }
    LBM_HD static constexpr int M(int k, int i) {
        const int x = D2Q9::ex(i), y = D2Q9::ey(i), n2 = x * x + y * y;
        return k == 0 ? 1
             : k == 1 ? -4 + 3 * n2
             : k == 2 ? (8 - 21 * n2 + 9 * n2 * n2) / 2
             : k == 3 ? x
             : k == 4 ? (-5 + 3 * n2) * x
             : k == 5 ? y
             : k == 6 ? (-5 + 3 * n2) * y
             : k == 7 ? x * x - y * y
             : x * y;
    }
    LBM_HD static void forward(const T (&d)[9], T (&m)[9]) {
#pragma unroll
        for (int k = 0; k < 9; k++) {
            T s = T(0);
#pragma unroll
            for (int i = 0; i < 9; i++) if (M(k, i) != 0) s += T(M(k, i)) * d[i];
            m[k] = s;
        }
    }
    LBM_HD static void backward(const T (&r)[9], T (&o)[9]) {
#pragma unroll
        for (int i = 0; i < 9; i++) {
            T s = T(0);
#pragma unroll
            for (int k = 0; k < 9; k++) if (M(k, i) != 0) s += T(M(k, i)) * r[k];
            o[i] = s;
        }
    }
};

// FORCE: 0 no body force, 1 Guo (eq. 17), 2 Exact Difference Method (eq. 18).
constexpr int FORCE_NONE = 0, FORCE_GUO = 1, FORCE_EDM = 2;
// MODEL: LBGK (Alg. 1 l.13) | MRT (eq. 4) | regularized LBGK | LBGK + Smagorinsky (eq. 8-9).
constexpr int MODEL_BGK = 0, MODEL_MRT = 1, MODEL_REG = 2, MODEL_LES = 3;

// ---- collision: h (pre-collision deviations) -> h* (post-collision), in place ---------------
// rho, drho = rho - 1, v = velocity entering f^eq and eq. (17) (reading A3), rv = rho v as formed
// from the moments (j + F/2, eq. 16), F = force density.  With FORCE_EDM v is the bare velocity u
// (reading A22), rv = rho u, and the routine adds f^eq(rho, u + F/rho) - f^eq(rho, u).
template <class L, typename T, int MODEL, int FORCE>
LBM_HD void collide(T (&h)[L::Q], T rho, T drho, const T (&v)[3], const T (&rv)[3], const T (&F)[3], const Relax<T> &rp) {
    constexpr int Q = L::Q;
    if constexpr (MODEL != MODEL_MRT) {
        // LBGK (Alg. 1 l.13) + eq. (17), evaluated per +/- pair of directions: with e_ibar = -e_i
        // the equilibrium and the source split into a part even in e_i (shared by the pair) and a
        // part odd in e_i (opposite signs), which halves the arithmetic per node.
        //
        // Round-off: a constant such as fl(omega w_i) carries the same rounding
        // error at every node and step; in fp32 that made sum_i e_i f_i^eq differ from rho u by a
        // fixed 6e-8 relative, i.e. a velocity drift of 7.6e-8 per step (1e-4 after 1300 steps on the
        // Taylor-Green case).  Therefore: the weights enter as the exact integers 36 w_i (powers
        // of two on all moving directions), omega / 36 multiplies the three per-node scalars as a
        // two-term sum hi + lo (rounding then depends on the node's data, not on a constant), and
        // the old value is scaled by keep = 1 - omega, which set_bgk makes exact for the omega in use.
        // relaxation constants: host-prepared (set_bgk) or, for the Smagorinsky model, per node
        T keep = rp.keep, om = rp.inv_tau, om36_hi = rp.om36_hi, om36_lo = rp.om36_lo;
        T sc36_hi = rp.sc36_hi, sc36_lo = rp.sc36_lo;
        if constexpr (MODEL == MODEL_REG || MODEL == MODEL_LES) {
            // non-equilibrium second moment sum_i e_ia e_ib (h_i - h_i^eq) = P_ab - (rho - 1) delta_ab / 3
            // - rho v_a v_b; it is Pi^neq of P:130 and Q of eq. (9) at once because sum_i f_i^neq = 0
            T Pi[6];
            second_moments<L, T>(h, Pi);
            const T third = drho * T(1.0 / 3.0);
            Pi[0] -= third + rho * v[0] * v[0];
            Pi[1] -= third + rho * v[1] * v[1];
            Pi[2] -= L::D == 3 ? third + rho * v[2] * v[2] : T(0);
            Pi[3] -= rho * v[0] * v[1];
            Pi[4] -= rho * v[1] * v[2];
            Pi[5] -= rho * v[0] * v[2];
            if constexpr (MODEL == MODEL_LES) {
                // eq. (9): tau = tau_0 + ( sqrt(tau_0^2 + 36 C_S^2 |Q|) - tau_0 ) / 2, |Q| = (Q_ab Q_ab)^(1/2)
                const T q2 = Pi[0] * Pi[0] + Pi[1] * Pi[1] + Pi[2] * Pi[2] +
                             T(2) * (Pi[3] * Pi[3] + Pi[4] * Pi[4] + Pi[5] * Pi[5]);
                const T tau = T(0.5) * (rp.tau0 + sqrt(rp.tau0 * rp.tau0 + rp.cs2x36 * sqrt(q2)));
                om = T(1) / tau;
                keep = T(1) - om;
                om36_hi = om * T(1.0 / 36.0); om36_lo = T(0);
                sc36_hi = (T(1) - T(0.5) * om) * T(1.0 / 36.0); sc36_lo = T(0);
            } else {
                // regularized: h* = keep f^reg + h^eq(u2), f^reg_i = 4.5 w_i (e_i.Pi.e_i - tr Pi / 3),
                // u2 = u + F / rho (the EDM increment; u2 = u without a force).  Reading A23.
                const T inv_rho = T(1) / rho;
                T u2[3], mo[3];
#pragma unroll
                for (int a = 0; a < 3; a++) {
                    u2[a] = FORCE ? v[a] + F[a] * inv_rho : v[a];
                    const T t = T(3) * (FORCE ? rv[a] + F[a] : rv[a]);
                    mo[a] = t * rp.i36_hi + t * rp.i36_lo;
                }
                const T vv2 = u2[0] * u2[0] + u2[1] * u2[1] + u2[2] * u2[2];
                const T b0 = drho - rho * (T(1.5) * vv2), q0 = T(4.5) * rho;
                const T k8 = keep * T(0.125);  // keep * 4.5 / 36
                const T tr3 = (Pi[0] + Pi[1] + Pi[2]) * T(1.0 / 3.0);
                const T base = (b0 * rp.i36_hi + b0 * rp.i36_lo) - k8 * tr3;
                const T r45 = q0 * rp.i36_hi + q0 * rp.i36_lo;
                h[0] = T(L::w36(0)) * base;
#pragma unroll
                for (int i = 1; i < Q; i++) {
                    if (i < L::opp(i)) {
                        const int j = L::opp(i);
                        const T wi = T(L::w36(i));
                        const T ev2 = e_dot<L, T>(i, u2);
                        const T odd = e_dot<L, T>(i, mo);
                        const T even = base + r45 * ev2 * ev2 + k8 * e_quad<L, T>(i, Pi);
                        h[i] = wi * (even + odd);
                        h[j] = wi * (even - odd);
                    }
                }
                return;
            }
        }
        if constexpr (FORCE == FORCE_EDM) {
            // h* = keep h + h^eq(u2) - keep h^eq(u), u2 = u + F/rho, in the same even/odd form:
            //   odd  = 3 e.(rho u2 - keep rho u) = 3 e.(omega rho u + F)   (momentum gains exactly F)
            //   even = omega drho - 1.5 rho (u2^2 - keep u^2) + 4.5 rho ((e.u2)^2 - keep (e.u)^2)
            const T inv_rho = T(1) / rho;
            T u2[3], mo[3];
#pragma unroll
            for (int a = 0; a < 3; a++) {
                u2[a] = v[a] + F[a] * inv_rho;
                const T t = T(3) * rv[a], f3 = T(3) * F[a];
                mo[a] = (t * om36_hi + t * om36_lo) + (f3 * rp.i36_hi + f3 * rp.i36_lo);
            }
            const T vv = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
            const T vv2 = u2[0] * u2[0] + u2[1] * u2[1] + u2[2] * u2[2];
            const T b0 = om * drho - rho * (T(1.5) * (vv2 - keep * vv)), q0 = T(4.5) * rho;
            const T base = b0 * rp.i36_hi + b0 * rp.i36_lo;
            const T r45 = q0 * rp.i36_hi + q0 * rp.i36_lo;
            h[0] = keep * h[0] + T(L::w36(0)) * base;
#pragma unroll
            for (int i = 1; i < Q; i++) {
                if (i < L::opp(i)) {
                    const int j = L::opp(i);
                    const T wi = T(L::w36(i));
                    const T ev = e_dot<L, T>(i, v), ev2 = e_dot<L, T>(i, u2);
                    const T odd = e_dot<L, T>(i, mo);
                    const T even = base + r45 * (ev2 * ev2 - keep * (ev * ev));
                    h[i] = keep * h[i] + wi * (even + odd);
                    h[j] = keep * h[j] + wi * (even - odd);
                }
            }
            return;
        }
        const T vv = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
        const T b0 = drho - rho * (T(1.5) * vv), q0 = T(4.5) * rho;
        const T base = b0 * om36_hi + b0 * om36_lo;
        const T r45 = q0 * om36_hi + q0 * om36_lo;
        // odd part: omega w_i 3 rho (e_i . v) = 36 w_i e_i . m3 with m3 = (omega / 12) * (rho v),
        // and rho v = j + F/2 is taken from the moments directly (no round trip through 1/rho),
        // so that sum_i e_i f_i^eq reproduces it up to unbiased rounding.
        // With a force the source of eq. (17) folds into the same two sums: the odd part gains
        // 3 e_i.F' and the even part 9 (e_i.v)(e_i.F') - 3 v.F', F' = (1 - omega/2) F / 36.
        T mo[3], F9[3] = {T(0), T(0), T(0)}, base_f = base;
#pragma unroll
        for (int a = 0; a < 3; a++) {
            const T t = T(3) * rv[a];
            mo[a] = t * om36_hi + t * om36_lo;
        }
        if constexpr (FORCE) {
            T vF = T(0);
#pragma unroll
            for (int a = 0; a < 3; a++) {
                const T Fs = F[a] * sc36_hi + F[a] * sc36_lo;
                mo[a] += T(3) * Fs;
                F9[a] = T(9) * Fs;
                vF += v[a] * Fs;
            }
            base_f = base - T(3) * vF;
        }
        h[0] = keep * h[0] + T(L::w36(0)) * base_f;
#pragma unroll
        for (int i = 1; i < Q; i++) {
            if (i < L::opp(i)) {
                const int j = L::opp(i);
                const T wi = T(L::w36(i));
                const T ev = e_dot<L, T>(i, v);
                const T odd = e_dot<L, T>(i, mo);
                T even;
                if constexpr (FORCE) even = base_f + ev * (r45 * ev + e_dot<L, T>(i, F9));
                else even = base_f + r45 * ev * ev;
                h[i] = keep * h[i] + wi * (even + odd);
                h[j] = keep * h[j] + wi * (even - odd);
            }
        }
    } else {
        T heq[Q];
        equilibrium_dev<L, T>(rho, drho, v, heq);
        T d[Q], m[Q];
#pragma unroll
        for (int i = 0; i < Q; i++) d[i] = heq[i] - h[i];
        Mrt<L, T>::forward(d, m);
#pragma unroll
        for (int k = 0; k < Q; k++) m[k] *= rp.cr[k];
        if constexpr (FORCE == FORCE_GUO) {
            T src[Q], ms[Q];
            guo_bracket<L, T>(v, F, src);
            Mrt<L, T>::forward(src, ms);
#pragma unroll
            for (int k = 0; k < Q; k++) m[k] += rp.cs[k] * ms[k];
        }
        Mrt<L, T>::backward(m, d);
#pragma unroll
        for (int i = 0; i < Q; i++) h[i] += d[i];
        if constexpr (FORCE == FORCE_EDM) {
            const T inv_rho = T(1) / rho;
            T u2[3], heq2[Q];
#pragma unroll
            for (int a = 0; a < 3; a++) u2[a] = v[a] + F[a] * inv_rho;
            equilibrium_dev<L, T>(rho, drho, u2, heq2);
#pragma unroll
            for (int i = 0; i < Q; i++) h[i] += heq2[i] - heq[i];
        }
    }
}

// Single-component node update: moments, F = rho g, v = j/rho + g/2 (eq. 16), collide.
template <class L, typename T, int MODEL, int FORCE>
LBM_HD void update_node(T (&h)[L::Q], const Relax<T> &rp) {
    constexpr int Q = L::Q;
    if constexpr (MODEL == MODEL_MRT && Mrt<L, T>::closed_form_meq) {
        // eq. (4) in moment space: m = M h once (it also yields rho - 1 and j), relax towards the
        // closed-form equilibrium moments, transform back the increment only.
        T m[Q];
        Mrt<L, T>::forward(h, m);
        const T drho = m[0], rho = T(1) + drho, inv_rho = T(1) / rho;
        T v[3], F[3];
#pragma unroll
        for (int a = 0; a < 3; a++) {
            const T ja = m[3 + 2 * a];
            F[a] = FORCE ? rho * rp.g[a] : T(0);
            v[a] = FORCE == FORCE_GUO ? (ja + T(0.5) * F[a]) * inv_rho : ja * inv_rho;
        }
        T q[Q];
        Mrt<L, T>::meq_dev(rho, drho, v, q);
#pragma unroll
        for (int k = 0; k < Q; k++) m[k] = rp.cr[k] * (q[k] - m[k]);
        if constexpr (FORCE == FORCE_EDM) {  // + M^-1 (m^eq(u + F/rho) - m^eq(u)), eq. (18)
            T u2[3], q2[Q];
#pragma unroll
            for (int a = 0; a < 3; a++) u2[a] = v[a] + F[a] * inv_rho;
            Mrt<L, T>::meq_dev(rho, drho, u2, q2);
#pragma unroll
            for (int k = 0; k < Q; k++) m[k] += rp.in[k] * (q2[k] - q[k]);
        }
        if constexpr (FORCE == FORCE_GUO) {
            T src[Q], ms[Q];
            guo_bracket<L, T>(v, F, src);
            Mrt<L, T>::forward(src, ms);
#pragma unroll
            for (int k = 0; k < Q; k++) m[k] += rp.cs[k] * ms[k];
        }
        T o[Q];
        Mrt<L, T>::backward(m, o);
#pragma unroll
        for (int i = 0; i < Q; i++) h[i] += o[i];
    } else {
        T drho, j[3];
        moments<L, T>(h, drho, j);
        const T rho = T(1) + drho, inv_rho = T(1) / rho;
        T v[3], rv[3], F[3];
#pragma unroll
        for (int a = 0; a < 3; a++) {
            F[a] = FORCE ? rho * rp.g[a] : T(0);
            rv[a] = FORCE == FORCE_GUO ? j[a] + T(0.5) * F[a] : j[a];
            v[a] = rv[a] * inv_rho;
        }
        collide<L, T, MODEL, FORCE>(h, rho, drho, v, rv, F, rp);
    }
}

// ---- node types that replace the collision (readings A20, A21) --------------------
// Full-way bounce-back wall node (Fig. 2 (1)): dry; the populations streamed into it are
// scattered back, h*_i = h_ibar, without relaxation.
template <class L, typename T> LBM_HD void fullway_reverse(T (&h)[L::Q]) {
#pragma unroll
    for (int i = 1; i < L::Q; i++)
        if (i < L::opp(i)) { const T t = h[i]; h[i] = h[L::opp(i)]; h[L::opp(i)] = t; }
}

// Equilibrium-velocity node: rho from the node's own incoming populations (the missing ones
// are bounce-back copies, supplied by the reflected-link rule), post-collision state f^eq(rho, u_bc).
template <class L, typename T> LBM_HD void velocity_node(T (&h)[L::Q], const T (&ubc)[3]) {
    T drho = h[0];
#pragma unroll
    for (int i = 1; i < L::Q; i++) drho += h[i];
    equilibrium_dev<L, T>(T(1) + drho, drho, ubc, h);
}

}  // namespace lbm
