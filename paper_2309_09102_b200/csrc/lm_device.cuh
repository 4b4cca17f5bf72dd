// lm_device.cuh -- per-waypoint device arithmetic of the batched LM pose refinement (sm_100a).
//
// One THREAD owns one waypoint block: its d x d damped normal equations are independent of every
// other waypoint (block-diagonal Jacobian), so all state lives in registers and all
// loops over joints are unrolled at compile time.  Every floating-point operation is written as
// an explicit round-to-nearest intrinsic (fmaf / __fmul_rn / __fadd_rn): the compiler may neither
// contract nor reassociate them, so a waypoint's bits do not depend on which kernel, launch
// geometry or batch it is evaluated in (bit-stability).
//
// The STRUCTURE of the kinematic chain (which joints are prismatic, which link twists are 0 or
// +-pi/2, which link offsets vanish) is a compile-time ChainSpec: for a registered robot the
// multiplications by 0 / +-1, the offset adds and every warp-uniform branch disappear from the
// instruction stream.  Skipping a term that is exactly zero (or multiplying by exactly +-1)
// leaves every result unchanged, so a specialised kernel returns the same values as the generic one.
//
// Step names S1..S9 follow DESIGN.md section 2.
#pragma once
#ifndef __CUDACC_RTC__
#include <cuda_runtime.h>
#include <stdint.h>
#else // run-time compilation (lm_jit.cu): NVRTC has the CUDA built-ins but no host headers
typedef signed char int8_t;
typedef unsigned char uint8_t;
typedef unsigned short uint16_t;
typedef int int32_t;
typedef unsigned int uint32_t;
typedef long long int64_t;
typedef unsigned long long uint64_t;
#endif

namespace lmk {

constexpr int MAX_DOF = 8;

// Chain constants, fp32, passed by value inside the kernel parameter block (constant bank).
struct KChain {
    float ca[MAX_DOF], sa[MAX_DOF];   // cos / sin alpha_{j-1}
    float a[MAX_DOF], d[MAX_DOF];     // a_{j-1}, d_j offset
    float toff[MAX_DOF];              // theta offset (revolute)
    float cth[MAX_DOF], sth[MAX_DOF]; // cos / sin of the fixed theta (prismatic)
    float lo[MAX_DOF], hi[MAX_DOF];   // joint limits, rounded inward to fp32
    float tool_p[3];
    float tool_R[9];                  // row-major
    uint32_t prismatic_mask;          // bit j: joint j prismatic
    uint32_t tool_has_rot;            // tool rotation != identity
};

// Compile-time structure of a chain.  generic = true: everything is decided at run time from
// KChain (warp-uniform branches).  Otherwise the masks say, per joint j (bit j):
struct ChainSpec {
    bool generic;
    int dof;
    uint32_t pris; // prismatic
    uint32_t al0;  // alpha == 0
    uint32_t alp;  // alpha == +pi/2  (ca = 0, sa = +1)
    uint32_t aln;  // alpha == -pi/2  (ca = 0, sa = -1)
    uint32_t a0;   // a == 0
    uint32_t d0;   // d offset == 0
    uint32_t t0;   // theta offset == 0
    bool tool_rot; // tool rotation != identity
    uint32_t tp0;  // bit i: tool_p[i] == 0
};

__host__ __device__ constexpr ChainSpec generic_spec(int d) { return ChainSpec{true, d, 0, 0, 0, 0, 0, 0, 0, true, 0}; }

__device__ __forceinline__ float mul(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float add(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float sub(float a, float b) { return __fsub_rn(a, b); }
__device__ __forceinline__ float fma_(float a, float b, float c) { return __fmaf_rn(a, b, c); }

// sin and cos of x for |x| < ~100 (joint angles are bounded by the joint limits).
// Cody-Waite reduction by pi/2 in two parts (FMA: the products are exact), then the classic single-precision minimax
// polynomials on [-pi/4, pi/4]; max error ~1 ulp.  FAST: the MUFU approximations (abs err ~5e-7).
template <bool FAST>
__device__ __forceinline__ void sincos_(float x, float &s, float &c) {
    if (FAST) {
        __sincosf(x, &s, &c);
        return;
    }
    const float magic = 12582912.0f;                     // 1.5 * 2^23: rounds to nearest integer
    float t = fma_(x, 0.636619772f, magic);              // x * 2/pi
    int qd = __float_as_int(t);                          // quadrant in the low mantissa bits
    float j = sub(t, magic);
    float r = fma_(j, -1.57079601e+00f, x);   // pi/2 = 1.57079601 + 3.13916473e-07 + 5.4e-15: the third part moves r by
    r = fma_(j, -3.13916473e-07f, r);         // < 2e-14 for the |j| <= 3 the joint limits allow and is dropped
    float r2 = mul(r, r);
    float ps = fma_(r2, -1.9515295891e-4f, 8.3321608736e-3f);
    ps = fma_(ps, r2, -1.6666654611e-1f);
    float sn = fma_(mul(r, r2), ps, r);
    float pc = fma_(r2, 2.443315711809948e-5f, -1.388731625493765e-3f);
    pc = fma_(pc, r2, 4.166664568298827e-2f);
    pc = fma_(pc, r2, -0.5f);
    float cs = fma_(pc, r2, 1.0f);
    float s0 = (qd & 1) ? cs : sn;
    float c0 = (qd & 1) ? sn : cs;
    s = __int_as_float(__float_as_int(s0) ^ ((qd & 2) << 30));
    c = __int_as_float(__float_as_int(c0) ^ (((qd + 1) & 2) << 30));
}

// theta = atan2(s, c) for s >= 0, theta in [0, pi].  Odd polynomial on [0, 1] (rel. err 1e-7,
// coefficients: csrc/gen_atan_coeffs.py) + the usual octant reflections.
__device__ __forceinline__ float atan2_pos(float s, float c) {
    float ac = fabsf(c);
    float mx = fmaxf(s, ac), mn = fminf(s, ac);
    float t = __fdividef(mn, fmaxf(mx, 1e-30f));
    float t2 = mul(t, t);
    float p = fma_(t2, 2.622244181e-03f, -1.513253432e-02f);
    p = fma_(p, t2, 4.112185538e-02f);
    p = fma_(p, t2, -7.366705686e-02f);
    p = fma_(p, t2, 1.057393178e-01f);
    p = fma_(p, t2, -1.418597549e-01f);
    p = fma_(p, t2, 1.999039650e-01f);
    p = fma_(p, t2, -3.333298564e-01f);
    float at = fma_(mul(p, t2), t, t);
    float th = (s > ac) ? sub(1.57079632679f, at) : at;
    return (c < 0.0f) ? sub(3.14159265359f, th) : th;
}

// atan2(y, x) in (-pi, pi]
__device__ __forceinline__ float atan2_full(float y, float x) { return copysignf(atan2_pos(fabsf(y), x), y); }

// Pose of one waypoint: everything the LM iteration needs from FK.
template <int D>
struct Pose {
    float Jv[D][3]; // linear part of Jacobian column j   (S3)
    float Jw[D][3]; // angular part = joint axis z_j (0 for prismatic)
    float r[6];     // residual (S2)
    float F;        // r . r
    float Ei[9];    // roll-pitch-yaw variant only: E(rpy)^-1 at this pose (row-major), d(rpy)/dq = E^-1 J_w
};

// w = Log(E)^vee for cos(theta) < -0.9 (theta > 154 deg: an IK seed on the wrong wrist flip; rare in the documented
// workloads).  There v = sin(theta) a is short and carries an absolute fp32 error of ~1e-7, so the direction v / |v|
// is off by 1e-7 / sin(theta) -- 3e-4 rad of residual at theta = pi - 1e-3, everything at theta = pi (at the switch,
// sin(theta) = 0.44, it is 6e-7).  The symmetric part stays well conditioned: E_ii = c + (1 - c) a_i^2 and
// E_mi + E_im = 2 (1 - c) a_m a_i with 1 - c > 1.9.
// Largest component a_m (>= 1/sqrt 3) from the diagonal, the other two from the off-diagonal sums divided by it
// (a square root of a small diagonal difference would lose half the digits), the overall sign from v.
__device__ __forceinline__ void log_far(const float (&X)[3], const float (&Y)[3], const float (&Z)[3],
                                        const float (&Rt)[3][3], const float (&v)[3], float cth, float theta,
                                        float (&w)[3]) {
    float E[3][3];
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int k = 0; k < 3; ++k)
            E[i][k] = fma_(Z[i], Rt[2][k], fma_(Y[i], Rt[1][k], mul(X[i], Rt[0][k])));
    const float inv = __fdividef(1.0f, sub(1.0f, cth));
    float d2[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) d2[i] = mul(sub(E[i][i], cth), inv);
    int m = 0;
    float dmax = d2[0];
    if (d2[1] > dmax) { dmax = d2[1]; m = 1; }
    if (d2[2] > dmax) { dmax = d2[2]; m = 2; }
    const float am = sqrtf(fmaxf(dmax, 0.25f));
    const float k = __fdividef(mul(0.5f, inv), am);
    float ax[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const float sym = (m == 0) ? add(E[0][i], E[i][0]) : (m == 1) ? add(E[1][i], E[i][1]) : add(E[2][i], E[i][2]);
        ax[i] = (i == m) ? am : mul(sym, k);
    }
    const float dt = fma_(ax[2], v[2], fma_(ax[1], v[1], mul(ax[0], v[0])));
    const float th = (dt < 0.f) ? -theta : theta;
#pragma unroll
    for (int i = 0; i < 3; ++i) w[i] = mul(th, ax[i]);
}

// Entries of the Jacobian that the chain STRUCTURE fixes to exactly 0 or exactly 1 (unweighted):
// bit 3 j + k of `zv` / `zw` = linear / angular component k of column j is 0, `ov` / `ow` likewise 1.
//   joint 0 with alpha = 0: z_0 = e_z and o_0 on the z axis  => revolute: Jw_0 = (0,0,1), Jv_0[2] = 0;
//                                                               prismatic: Jv_0 = (0,0,1), Jw_0 = 0
//   joint 1 after such a joint 0: alpha = +-pi/2 => z_1 = -+Y_0 with Y_0[2] = 0; alpha = 0 => z_1 = e_z
//   any prismatic joint: Jw_j = 0.
// Terms with a known 0 are skipped and multiplications by a known 1 become additions in the dot
// products below: the results equal the generic kernel's up to the sign of zero.
struct JKnown { uint32_t zv, zw, ov, ow; };
__host__ __device__ constexpr JKnown jknown(const ChainSpec S, bool weighted, bool rpy = false) {
    JKnown K{0, 0, 0, 0};
    if (S.generic) return K;
    for (int j = 0; j < S.dof; ++j)
        if ((S.pris >> j) & 1u) K.zw |= 7u << (3 * j);
    const bool z0_ez = (S.al0 & 1u) != 0;
    if (z0_ez) {
        if (S.pris & 1u) { K.zv |= 3u; K.ov |= 4u; }
        else { K.zw |= 3u; K.ow |= 4u; K.zv |= 4u; }
        if (S.dof > 1) {
            const bool p1 = (S.pris & 2u) != 0;
            if ((S.al0 >> 1) & 1u) { // z_1 = e_z as well
                if (p1) { K.zv |= 3u << 3; K.ov |= 4u << 3; }
                else { K.zw |= 3u << 3; K.ow |= 4u << 3; }
                // Jv_1[2] = 0 needs o_1 on the z axis too (a_1 = 0): not assumed
            } else if (((S.alp | S.aln) >> 1) & 1u) { // z_1 = -+Y_0, Y_0[2] = 0
                if (p1) K.zv |= 4u << 3;
                else K.zw |= 4u << 3;
            }
        }
    }
    if (weighted) { K.ov = 0; K.ow = 0; } // a known 1 becomes the weight
    if (rpy) { K.zw = 0; K.ow = 0; }      // the angular rows are E^-1 J_w: nothing is known about them
    return K;
}

template <bool WEIGHTED, typename SpecT, bool RPY = false>
struct JK {
    static constexpr JKnown K = jknown(SpecT::spec, WEIGHTED, RPY);
    __device__ __forceinline__ static constexpr bool zero(int j, int k) { return (((k < 3 ? K.zv : K.zw) >> (3 * j + (k < 3 ? k : k - 3))) & 1u) != 0; }
    __device__ __forceinline__ static constexpr bool one(int j, int k) { return (((k < 3 ? K.ov : K.ow) >> (3 * j + (k < 3 ? k : k - 3))) & 1u) != 0; }
};
struct NoSpec { static constexpr ChainSpec spec = generic_spec(MAX_DOF); };

// S3: geometric Jacobian (DESIGN R3): revolute [z x (p - o); z], prismatic [z; 0], from the joint axes z_j
// (src.Jw) and frame origins o_j (src.Jv) that FK retained; dst may be src.
template <int D, bool WEIGHTED, typename SpecT, bool RPY = false>
__device__ __forceinline__ void finish_jacobian(const KChain &ch, const Pose<D> &src, const float (&p)[3], float w_pos,
                                                float w_rot, Pose<D> &dst) {
    constexpr ChainSpec S = SpecT::spec;
#pragma unroll
    for (int j = 0; j < D; ++j) {
        const bool pris = S.generic ? (((ch.prismatic_mask >> j) & 1u) != 0) : (((S.pris >> j) & 1u) != 0);
        const float z[3] = {src.Jw[j][0], src.Jw[j][1], src.Jw[j][2]};
        if (!pris) {
            // z x e with the components of z the chain structure fixes to 0 / 1 folded away (jknown)
            using K = JK<false, SpecT>;
            const float e[3] = {sub(p[0], src.Jv[j][0]), sub(p[1], src.Jv[j][1]), sub(p[2], src.Jv[j][2])};
            float c[3];
#pragma unroll
            for (int i = 0; i < 3; ++i) { // c_i = z_a e_b - z_b e_a, (a, b) = (i+1, i+2) mod 3, as fma(z_a, e_b, -z_b * e_a)
                const int a = (i + 1) % 3, b = (i + 2) % 3;
                const bool za0 = K::zero(j, 3 + a), za1 = K::one(j, 3 + a), zb0 = K::zero(j, 3 + b), zb1 = K::one(j, 3 + b);
                const float inner = zb0 ? 0.f : zb1 ? -e[a] : mul(-z[b], e[a]);
                c[i] = za0 ? inner : za1 ? (zb0 ? e[b] : add(e[b], inner)) : (zb0 ? mul(z[a], e[b]) : fma_(z[a], e[b], inner));
            }
#pragma unroll
            for (int i = 0; i < 3; ++i) {
                dst.Jv[j][i] = c[i];
                // roll-pitch-yaw variant: the angular rows become d(rpy)/dq = E^-1 z_j
                dst.Jw[j][i] = RPY ? fma_(src.Ei[3 * i + 2], z[2], fma_(src.Ei[3 * i + 1], z[1], mul(src.Ei[3 * i], z[0]))) : z[i];
            }
        } else {
#pragma unroll
            for (int i = 0; i < 3; ++i) { dst.Jv[j][i] = z[i]; dst.Jw[j][i] = 0.f; }
        }
        if (WEIGHTED) {
#pragma unroll
            for (int i = 0; i < 3; ++i) { dst.Jv[j][i] = mul(w_pos, dst.Jv[j][i]); dst.Jw[j][i] = mul(w_rot, dst.Jw[j][i]); }
        }
    }
}

// S1 + S2 + S3: serial-chain FK (modified DH, DESIGN R1), pose residual against the target
// (p_t, R_t given as COLUMNS Rt[k] = k-th column), geometric Jacobian from the retained joint axes.
//   A_j = Rot_x(alpha) Trans_x(a) Rot_z(theta) Trans_z(d);  frame columns X, Y, Z and origin o.
//   WITH_JAC = false: S3 is left to the caller (finish_jacobian); P.Jw / P.Jv then hold z_j / o_j and
//   frame_p (nullable) receives the flange position.
//   sink(j, X, Y, Z, o) is called with the frame of every link right after joint j (collision capsules ride on
//   link frames, lm_traj.cuh); the default does nothing.
struct NoFrameSink {
    __device__ __forceinline__ void operator()(int, const float (&)[3], const float (&)[3], const float (&)[3], const float (&)[3]) const {}
};
//   RPY = true (variant): the rotational residual is the wrapped element-wise difference of
//   roll, pitch, yaw (PAPER.md:L47, L115-117 read literally) against `trpy` = rpy of the target.
template <int D, bool FAST, bool WEIGHTED, typename SpecT, bool WITH_JAC = true, typename Sink = NoFrameSink, bool RPY = false>
__device__ __forceinline__ void eval_pose(const KChain &ch, const float (&q)[D], const float (&pt)[3],
                                          const float (&Rt)[3][3], float w_pos, float w_rot,
                                          Pose<D> &P, float *p_out, float (*R_out)[3], float *frame_p = nullptr,
                                          const Sink &sink = Sink(), const float *trpy = nullptr) {
    constexpr ChainSpec S = SpecT::spec;
    float X[3], Y[3], Z[3], o[3];
#pragma unroll
    for (int j = 0; j < D; ++j) {
        const bool pris = S.generic ? (((ch.prismatic_mask >> j) & 1u) != 0) : (((S.pris >> j) & 1u) != 0);
        const bool al0 = !S.generic && ((S.al0 >> j) & 1u), alp = !S.generic && ((S.alp >> j) & 1u),
                   aln = !S.generic && ((S.aln >> j) & 1u);
        const bool a_zero = !S.generic && ((S.a0 >> j) & 1u), d_zero = !S.generic && ((S.d0 >> j) & 1u) && !pris,
                   t_zero = !S.generic && ((S.t0 >> j) & 1u);
        float s, c, dj = 0.f;
        if (!pris) {
            sincos_<FAST>(t_zero ? q[j] : add(q[j], ch.toff[j]), s, c);
            if (!d_zero) dj = ch.d[j];
        } else {
            s = ch.sth[j];
            c = ch.cth[j];
            dj = add(ch.d[j], q[j]);
        }
        const float ca = ch.ca[j], sa = ch.sa[j], aj = ch.a[j];
        if (j == 0) {
            // base frame = identity: Y' = (0, ca, sa), Z' = (0, -sa, ca), o' = (a, 0, 0)
            float y1[3], z1[3];
            y1[0] = 0.f; z1[0] = 0.f;
            if (al0)      { y1[1] = 1.f; y1[2] = 0.f;  z1[1] = 0.f;  z1[2] = 1.f; }
            else if (alp) { y1[1] = 0.f; y1[2] = 1.f;  z1[1] = -1.f; z1[2] = 0.f; }
            else if (aln) { y1[1] = 0.f; y1[2] = -1.f; z1[1] = 1.f;  z1[2] = 0.f; }
            else          { y1[1] = ca;  y1[2] = sa;   z1[1] = -sa;  z1[2] = ca; }
            X[0] = c;  X[1] = (al0 ? s : (alp || aln) ? 0.f : mul(s, y1[1]));  X[2] = (al0 ? 0.f : alp ? s : aln ? -s : mul(s, y1[2]));
            Y[0] = -s; Y[1] = (al0 ? c : (alp || aln) ? 0.f : mul(c, y1[1]));  Y[2] = (al0 ? 0.f : alp ? c : aln ? -c : mul(c, y1[2]));
            o[0] = a_zero ? 0.f : aj;
            o[1] = (d_zero || al0) ? 0.f : mul(dj, z1[1]);
            o[2] = d_zero ? 0.f : (al0 ? dj : (alp || aln) ? 0.f : mul(dj, z1[2]));
#pragma unroll
            for (int i = 0; i < 3; ++i) { Z[i] = z1[i]; P.Jw[j][i] = z1[i]; P.Jv[j][i] = o[i]; }
            sink(j, X, Y, Z, o);
            continue;
        }
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            float y1, z1;
            if (al0)      { y1 = Y[i];  z1 = Z[i]; }                       // Rot_x(0)
            else if (alp) { y1 = Z[i];  z1 = -Y[i]; }                      // Rot_x(+pi/2)
            else if (aln) { y1 = -Z[i]; z1 = Y[i]; }                       // Rot_x(-pi/2)
            else {
                y1 = fma_(sa, Z[i], mul(ca, Y[i]));                         // Y' =  ca Y + sa Z
                z1 = fma_(ca, Z[i], mul(-sa, Y[i]));                        // Z' = -sa Y + ca Z
            }
            const float o1 = a_zero ? o[i] : fma_(aj, X[i], o[i]);          // Trans_x(a)
            const float x2 = fma_(s, y1, mul(c, X[i]));                     // Rot_z: X'' =  c X + s Y'
            const float y2 = fma_(c, y1, mul(-s, X[i]));                    //        Y'' = -s X + c Y'
            o[i] = d_zero ? o1 : fma_(dj, z1, o1);                          // Trans_z(d)
            X[i] = x2; Y[i] = y2; Z[i] = z1;
            P.Jw[j][i] = z1;                                                // joint axis z_j
            P.Jv[j][i] = o[i];                                              // frame origin o_j (-> J_v below)
        }
        sink(j, X, Y, Z, o);
    }
    // flange: p = o + R tool_p ;  R_ee = R R_tool
    float p[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        float t = o[i];
        if (S.generic || !(S.tp0 & 1u)) t = fma_(X[i], ch.tool_p[0], t);
        if (S.generic || !(S.tp0 & 2u)) t = fma_(Y[i], ch.tool_p[1], t);
        if (S.generic || !(S.tp0 & 4u)) t = fma_(Z[i], ch.tool_p[2], t);
        p[i] = t;
    }
    if (S.generic ? (ch.tool_has_rot != 0) : S.tool_rot) {
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            float x = X[i], y = Y[i], z = Z[i];
            X[i] = fma_(z, ch.tool_R[6], fma_(y, ch.tool_R[3], mul(x, ch.tool_R[0])));
            Y[i] = fma_(z, ch.tool_R[7], fma_(y, ch.tool_R[4], mul(x, ch.tool_R[1])));
            Z[i] = fma_(z, ch.tool_R[8], fma_(y, ch.tool_R[5], mul(x, ch.tool_R[2])));
        }
    }
    if (p_out) {
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            p_out[i] = p[i];
            R_out[i][0] = X[i]; R_out[i][1] = Y[i]; R_out[i][2] = Z[i];
        }
    }

    float w[3];
    if (RPY) {
        // R = Rz(yaw) Ry(pitch) Rx(roll): R31 = X[2] = -sin(pitch), R32 = Y[2], R33 = Z[2], R11 = X[0], R21 = X[1]
        const float cp = sqrtf(fma_(X[1], X[1], mul(X[0], X[0])));
        const float a[3] = {atan2_full(Y[2], Z[2]), atan2_full(-X[2], cp), atan2_full(X[1], X[0])};
#pragma unroll
        for (int i = 0; i < 3; ++i) { // wrap to (-pi, pi]
            const float dlt = sub(a[i], trpy[i]);
            const float k = rintf(mul(dlt, 0.159154943f));
            w[i] = fma_(k, -1.74845553e-07f, fma_(k, -6.28318548f, dlt)); // 2 pi = 6.28318548 - 1.74845553e-07
        }
        // E^-1 = 1/cp [[cy, sy, 0], [-sy cp, cy cp, 0], [cy sp, sy sp, cp]]
        const float icp = __fdividef(1.0f, cp);
        const float cy = mul(X[0], icp), sy = mul(X[1], icp), tp_ = mul(-X[2], icp);
        P.Ei[0] = mul(cy, icp); P.Ei[1] = mul(sy, icp); P.Ei[2] = 0.f;
        P.Ei[3] = -sy;          P.Ei[4] = cy;           P.Ei[5] = 0.f;
        P.Ei[6] = mul(cy, tp_); P.Ei[7] = mul(sy, tp_); P.Ei[8] = 1.f;
    } else {
    // S2: E = R_ee R_t^T = sum_k a_k b_k^T (a_k, b_k = k-th columns);
    //     vee(antisym E) = 1/2 sum_k b_k x a_k,  tr E = sum_k a_k . b_k          (DESIGN R2)
    float v[3], tr;
    {
        const float *A0 = X, *A1 = Y, *A2 = Z;
        const float *B0 = Rt[0], *B1 = Rt[1], *B2 = Rt[2];
#define LM_CROSS_ACC(i, i1, i2)                                                                       \
    v[i] = fma_(B2[i1], A2[i2], fma_(-B2[i2], A2[i1],                                                 \
           fma_(B1[i1], A1[i2], fma_(-B1[i2], A1[i1], fma_(B0[i1], A0[i2], mul(-B0[i2], A0[i1]))))));
        LM_CROSS_ACC(0, 1, 2)
        LM_CROSS_ACC(1, 2, 0)
        LM_CROSS_ACC(2, 0, 1)
#undef LM_CROSS_ACC
        tr = fma_(A2[2], B2[2], fma_(A2[1], B2[1], fma_(A2[0], B2[0],
             fma_(A1[2], B1[2], fma_(A1[1], B1[1], fma_(A1[0], B1[0],
             fma_(A0[2], B0[2], fma_(A0[1], B0[1], mul(A0[0], B0[0])))))))));
    }
#pragma unroll
    for (int i = 0; i < 3; ++i) v[i] = mul(0.5f, v[i]);
    const float cth = fma_(0.5f, tr, -0.5f);
    const float s2 = fma_(v[2], v[2], fma_(v[1], v[1], mul(v[0], v[0])));
    const float sn = sqrtf(s2);
    const float theta = atan2_pos(sn, cth);
    // theta / s; the small-angle series 1 + s^2/6 takes over below s = 1e-4
    const float scale = (sn < 1e-4f) ? fma_(s2, 0.166666667f, 1.0f) : __fdividef(theta, sn);
    w[0] = mul(scale, v[0]); w[1] = mul(scale, v[1]); w[2] = mul(scale, v[2]);
    if (cth < -0.9f) log_far(X, Y, Z, Rt, v, cth, theta, w);
    }
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const float rp = sub(p[i], pt[i]);
        P.r[i] = WEIGHTED ? mul(w_pos, rp) : rp;
        P.r[3 + i] = WEIGHTED ? mul(w_rot, w[i]) : w[i];
    }
    P.F = fma_(P.r[5], P.r[5], fma_(P.r[4], P.r[4], fma_(P.r[3], P.r[3],
          fma_(P.r[2], P.r[2], fma_(P.r[1], P.r[1], mul(P.r[0], P.r[0]))))));

    if (frame_p) {
#pragma unroll
        for (int i = 0; i < 3; ++i) frame_p[i] = p[i];
    }
    if (WITH_JAC) finish_jacobian<D, WEIGHTED, SpecT, RPY>(ch, P, p, w_pos, w_rot, P);
}

template <int D>
__device__ __forceinline__ float jentry(const Pose<D> &P, int j, int k) { return k < 3 ? P.Jv[j][k] : P.Jw[j][k - 3]; }

// init + sum_k J[k][i] J[k][j] in the order k = 0..5 (rows 0..2 linear, 3..5 angular); HAVE = false: no init term
template <int D, bool WEIGHTED, typename SpecT, bool HAVE, bool RPY = false>
__device__ __forceinline__ float coldot_k(const Pose<D> &P, int i, int j, float init) {
    using K = JK<WEIGHTED, SpecT, RPY>;
    float acc = init;
    bool have = HAVE;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        if (K::zero(i, k) || K::zero(j, k)) continue;
        const float a = jentry<D>(P, i, k), b = jentry<D>(P, j, k);
        const bool oi = K::one(i, k), oj = K::one(j, k);
        if (oi && oj) acc = have ? add(acc, 1.f) : 1.f;
        else if (oi) acc = have ? add(acc, b) : b;
        else if (oj) acc = have ? add(acc, a) : a;
        else acc = have ? fma_(a, b, acc) : mul(a, b);
        have = true;
    }
    return have ? acc : 0.f;
}
// sum_k J[k][i] t[k]
template <int D, bool WEIGHTED, typename SpecT, bool RPY = false>
__device__ __forceinline__ float colvec_k(const Pose<D> &P, int i, const float (&t)[6]) {
    using K = JK<WEIGHTED, SpecT, RPY>;
    float acc = 0.f;
    bool have = false;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        if (K::zero(i, k)) continue;
        const float a = jentry<D>(P, i, k);
        if (K::one(i, k)) acc = have ? add(acc, t[k]) : t[k];
        else acc = have ? fma_(a, t[k], acc) : mul(a, t[k]);
        have = true;
    }
    return have ? acc : 0.f;
}
// structure-agnostic forms (trajectory-level kernels)
template <int D>
__device__ __forceinline__ float coldot(const Pose<D> &P, int i, int j) { return coldot_k<D, false, NoSpec, false>(P, i, j, 0.f); }
template <int D>
__device__ __forceinline__ float colvec(const Pose<D> &P, int i, const float (&t)[6]) { return colvec_k<D, false, NoSpec>(P, i, t); }

// x = (L L^T)^-1 b with L's strictly-lower part in L and 1/diag in invd
template <int D>
__device__ __forceinline__ void chol_solve(const float (&L)[D][D], const float (&invd)[D],
                                           const float (&b)[D], float (&x)[D]) {
    float y[D];
#pragma unroll
    for (int i = 0; i < D; ++i) {
        float s = b[i];
#pragma unroll
        for (int j = 0; j < i; ++j) s = fma_(-L[i][j], y[j], s);
        y[i] = mul(s, invd[i]);
    }
#pragma unroll
    for (int i = D - 1; i >= 0; --i) {
        float s = y[i];
#pragma unroll
        for (int j = i + 1; j < D; ++j) s = fma_(-L[j][i], x[j], s);
        x[i] = mul(s, invd[i]);
    }
}

// S4 + S5: A = J^T J + lambda I, g = J^T r, in-register Cholesky A = L L^T, delta = -A^-1 g,
// then `refine` steps of iterative refinement with the semi-normal residual
//   rho = -J^T (r + J delta) - lambda delta,  delta += A^-1 rho                     (DESIGN R4)
// which removes the 1/lambda amplification of fp32 rounding along the self-motion direction.
// Returns false on a non-positive pivot or a non-finite step (=> the iteration is a reject).
// REFINE >= 0: the number of refinement steps is a compile-time constant (the loop and its counter disappear and the
// scheduler sees one block); REFINE = -1: the run-time argument `refine`.  Same operations either way.
template <int D, bool WEIGHTED, typename SpecT, bool RPY = false, int REFINE = -1>
__device__ __forceinline__ bool lm_delta(const Pose<D> &P, float lam, int refine, float (&delta)[D]) {
    using K = JK<WEIGHTED, SpecT, RPY>;
    float L[D][D], invd[D], g[D];
#pragma unroll
    for (int i = 0; i < D; ++i) {
#pragma unroll
        for (int j = 0; j < i; ++j) L[i][j] = coldot_k<D, WEIGHTED, SpecT, false, RPY>(P, i, j, 0.f);
        L[i][i] = coldot_k<D, WEIGHTED, SpecT, true, RPY>(P, i, i, lam); // lambda folded into the first FMA of the diagonal
        g[i] = -colvec_k<D, WEIGHTED, SpecT, RPY>(P, i, P.r);
    }
    bool ok = true;
#pragma unroll
    for (int k = 0; k < D; ++k) {
        const float piv = L[k][k];
        ok = ok && (piv > 0.f);
        const float id = rsqrtf(piv);   // MUFU.RSQ (built with -ftz=true); pivots are >= ~lambda_min
        invd[k] = id;
#pragma unroll
        for (int i = k + 1; i < D; ++i) L[i][k] = mul(L[i][k], id);
#pragma unroll
        for (int j = k + 1; j < D; ++j)
#pragma unroll
            for (int i = j; i < D; ++i) L[i][j] = fma_(-L[i][k], L[j][k], L[i][j]);
    }
    chol_solve<D>(L, invd, g, delta);
    const int nref = REFINE >= 0 ? REFINE : refine;
#pragma unroll
    for (int it = 0; it < nref; ++it) {
        float t[6], rho[D], e[D];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            float sv = P.r[k], sw = P.r[3 + k];
#pragma unroll
            for (int j = 0; j < D; ++j) {
                if (!K::zero(j, k)) sv = K::one(j, k) ? add(sv, delta[j]) : fma_(P.Jv[j][k], delta[j], sv);
                if (!K::zero(j, 3 + k)) sw = K::one(j, 3 + k) ? add(sw, delta[j]) : fma_(P.Jw[j][k], delta[j], sw);
            }
            t[k] = sv;
            t[3 + k] = sw;
        }
#pragma unroll
        for (int i = 0; i < D; ++i) rho[i] = -fma_(lam, delta[i], colvec_k<D, WEIGHTED, SpecT, RPY>(P, i, t));
        chol_solve<D>(L, invd, rho, e);
#pragma unroll
        for (int i = 0; i < D; ++i) delta[i] = add(delta[i], e[i]);
    }
    float asum = 0.f;
#pragma unroll
    for (int i = 0; i < D; ++i) asum = add(asum, fabsf(delta[i]));
    return ok && (asum < 1e30f);
}

// ---- packed form of S4 + S5 (sm_100a FFMA2 / FMUL2: two fp32 operations per instruction, each IEEE round-to-nearest).
// Layout: the Jacobian in PAIRS OF COLUMNS, Jp[k][c] = (J[k][2c], J[k][2c+1]) (row k of 6, pad column = 0 when D is
// odd), and the lower triangle of A = J^T J + lambda I as column vectors paired along the row index,
// Ap[c][j] = (A[2c][j], A[2c+1][j]) for 2c+1 >= j.  Every entry goes through the same sequence of fused operations as
// in lm_delta (sum over k = 0..5, right-looking Cholesky, forward substitution by columns), so the step has the same
// bits up to the sign of zero; the extra lane of a boundary pair (a row above the diagonal, the pad row) is never read.
using f2 = float2;
__device__ __forceinline__ f2 bc2(float s) { return make_float2(s, s); }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ f2 add2(f2 a, f2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ f2 neg2(f2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ float lane2(f2 a, int l) { return l ? a.y : a.x; }

// x = (L L^T)^-1 b: forward substitution by columns on pairs (bp is consumed), backward substitution on scalars
template <int D>
__device__ __forceinline__ void chol_solve_p(const f2 (&Lp)[(D + 1) / 2][D], const float (&invd)[D], f2 (&bp)[(D + 1) / 2],
                                             float (&x)[D]) {
    constexpr int NP = (D + 1) / 2;
    float y[D];
#pragma unroll
    for (int j = 0; j < D; ++j) {
        y[j] = mul(lane2(bp[j / 2], j & 1), invd[j]);
#pragma unroll
        for (int c = (j + 1) / 2; c < NP; ++c) bp[c] = fma2(neg2(Lp[c][j]), bc2(y[j]), bp[c]);
    }
#pragma unroll
    for (int i = D - 1; i >= 0; --i) {
        float s = y[i];
#pragma unroll
        for (int j = i + 1; j < D; ++j) s = fma_(-lane2(Lp[j / 2][i], j & 1), x[j], s);
        x[i] = mul(s, invd[i]);
    }
}

template <int D, bool WEIGHTED, typename SpecT, bool RPY = false>
__device__ __forceinline__ bool lm_delta_p(const Pose<D> &P, float lam, int refine, float (&delta)[D]) {
    using K = JK<WEIGHTED, SpecT, RPY>;
    constexpr int NP = (D + 1) / 2;
    f2 Jp[6][NP];
#pragma unroll
    for (int k = 0; k < 6; ++k)
#pragma unroll
        for (int c = 0; c < NP; ++c) Jp[k][c] = make_float2(jentry<D>(P, 2 * c, k), 2 * c + 1 < D ? jentry<D>(P, 2 * c + 1, k) : 0.f);
    f2 Ap[NP][D], gp[NP];
#pragma unroll
    for (int j = 0; j < D; ++j)
#pragma unroll
        for (int c = j / 2; c < NP; ++c) {
            f2 a = make_float2(2 * c == j ? lam : 0.f, 2 * c + 1 == j ? lam : 0.f);
#pragma unroll
            for (int k = 0; k < 6; ++k) {
                if (K::zero(j, k)) continue;
                a = fma2(Jp[k][c], bc2(jentry<D>(P, j, k)), a);
            }
            Ap[c][j] = a;
        }
#pragma unroll
    for (int c = 0; c < NP; ++c) {
        f2 a = make_float2(0.f, 0.f);
#pragma unroll
        for (int k = 0; k < 6; ++k) a = fma2(Jp[k][c], bc2(P.r[k]), a);
        gp[c] = neg2(a);
    }
    float invd[D];
    bool ok = true;
#pragma unroll
    for (int k = 0; k < D; ++k) {
        const float piv = lane2(Ap[k / 2][k], k & 1);
        ok = ok && (piv > 0.f);
        const float id = rsqrtf(piv);
        invd[k] = id;
#pragma unroll
        for (int c = (k + 1) / 2; c < NP; ++c) Ap[c][k] = mul2(Ap[c][k], bc2(id));
#pragma unroll
        for (int j = k + 1; j < D; ++j) {
            const float b = lane2(Ap[j / 2][k], j & 1);
#pragma unroll
            for (int c = j / 2; c < NP; ++c) Ap[c][j] = fma2(neg2(Ap[c][k]), bc2(b), Ap[c][j]);
        }
    }
    chol_solve_p<D>(Ap, invd, gp, delta);
    for (int it = 0; it < refine; ++it) {
        float t[6], e[D];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            float sv = P.r[k], sw = P.r[3 + k];
#pragma unroll
            for (int j = 0; j < D; ++j) {
                if (!K::zero(j, k)) sv = K::one(j, k) ? add(sv, delta[j]) : fma_(P.Jv[j][k], delta[j], sv);
                if (!K::zero(j, 3 + k)) sw = K::one(j, 3 + k) ? add(sw, delta[j]) : fma_(P.Jw[j][k], delta[j], sw);
            }
            t[k] = sv;
            t[3 + k] = sw;
        }
        f2 rp[NP];
#pragma unroll
        for (int c = 0; c < NP; ++c) {
            f2 a = make_float2(0.f, 0.f);
#pragma unroll
            for (int k = 0; k < 6; ++k) a = fma2(Jp[k][c], bc2(t[k]), a);
            rp[c] = neg2(fma2(bc2(lam), make_float2(delta[2 * c], 2 * c + 1 < D ? delta[2 * c + 1] : 0.f), a));
        }
        chol_solve_p<D>(Ap, invd, rp, e);
#pragma unroll
        for (int i = 0; i < D; ++i) delta[i] = add(delta[i], e[i]);
    }
    float asum = 0.f;
#pragma unroll
    for (int i = 0; i < D; ++i) asum = add(asum, fabsf(delta[i]));
    return ok && (asum < 1e30f);
}

// ---- lane-group form of S4 + S5 (BASELINE.json north_star: "one warp or thread group per waypoint block ... warp-shuffle
// reductions for J^T J / J^T r"; measured against the one-thread form in DESIGN.md section 7): G = 2 or 4 adjacent
// lanes share one waypoint.  FK, the Jacobian, the Cholesky factorisation and the triangular solves are replicated on
// the G lanes (a serial chain and a 7 x 7 triangle do not split without per-step exchanges); the sums over the six rows
// of J -- J^T J, J^T r and J^T t of the refinement -- are split by rows (lane g takes rows g, g + G, ...) and closed with
// an xor butterfly, which leaves bit-identical totals on every lane of the group, so the G lanes take the same decisions.
// The summation order differs from lm_delta, so results agree with the one-thread kernel to rounding, not bitwise.
template <int G>
__device__ __forceinline__ float group_sum(float v) {
#pragma unroll
    for (int o = 1; o < G; o <<= 1) v = add(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
template <int D, int G>
__device__ __forceinline__ bool lm_delta_lg(const Pose<D> &P, float lam, int refine, int g, float (&delta)[D]) {
    static_assert(G == 2 || G == 4, "lane groups of 2 or 4");
    constexpr int R = (6 + G - 1) / G; // rows per lane
    float Jh[D][R], rh[R];
#pragma unroll
    for (int m = 0; m < R; ++m) {
        float rv = 0.f;
#pragma unroll
        for (int gg = 0; gg < G; ++gg)
            if (gg + G * m < 6) rv = (g == gg) ? P.r[gg + G * m] : rv;
        rh[m] = rv;
#pragma unroll
        for (int j = 0; j < D; ++j) {
            float v = 0.f;
#pragma unroll
            for (int gg = 0; gg < G; ++gg)
                if (gg + G * m < 6) v = (g == gg) ? jentry<D>(P, j, gg + G * m) : v;
            Jh[j][m] = v;
        }
    }
    float L[D][D], invd[D], gv[D];
#pragma unroll
    for (int i = 0; i < D; ++i) {
#pragma unroll
        for (int j = 0; j <= i; ++j) {
            float a = mul(Jh[i][0], Jh[j][0]);
#pragma unroll
            for (int m = 1; m < R; ++m) a = fma_(Jh[i][m], Jh[j][m], a);
            a = group_sum<G>(a);
            L[i][j] = (i == j) ? add(a, lam) : a;
        }
        float a = mul(Jh[i][0], rh[0]);
#pragma unroll
        for (int m = 1; m < R; ++m) a = fma_(Jh[i][m], rh[m], a);
        gv[i] = -group_sum<G>(a);
    }
    bool ok = true;
#pragma unroll
    for (int k = 0; k < D; ++k) {
        const float piv = L[k][k];
        ok = ok && (piv > 0.f);
        const float id = rsqrtf(piv);
        invd[k] = id;
#pragma unroll
        for (int i = k + 1; i < D; ++i) L[i][k] = mul(L[i][k], id);
#pragma unroll
        for (int j = k + 1; j < D; ++j)
#pragma unroll
            for (int i = j; i < D; ++i) L[i][j] = fma_(-L[i][k], L[j][k], L[i][j]);
    }
    chol_solve<D>(L, invd, gv, delta);
    for (int it = 0; it < refine; ++it) {
        float th[R], rho[D], e[D];
#pragma unroll
        for (int m = 0; m < R; ++m) {
            float sv = rh[m];
#pragma unroll
            for (int j = 0; j < D; ++j) sv = fma_(Jh[j][m], delta[j], sv);
            th[m] = sv;
        }
#pragma unroll
        for (int i = 0; i < D; ++i) {
            float a = mul(Jh[i][0], th[0]);
#pragma unroll
            for (int m = 1; m < R; ++m) a = fma_(Jh[i][m], th[m], a);
            rho[i] = -fma_(lam, delta[i], group_sum<G>(a));
        }
        chol_solve<D>(L, invd, rho, e);
#pragma unroll
        for (int i = 0; i < D; ++i) delta[i] = add(delta[i], e[i]);
    }
    float asum = 0.f;
#pragma unroll
    for (int i = 0; i < D; ++i) asum = add(asum, fabsf(delta[i]));
    return ok && (asum < 1e30f);
}

// The same step in its DUAL form (SURVEY section 8f NEXT-4 i, a disclosed variant):
//   delta = -J^T (J J^T + lambda I_6)^-1 r,
// identical to -(J^T J + lambda I_d)^-1 J^T r in exact arithmetic (push-through identity; the oracle pins
// it, tests/test_oracle_pins.py P5).  6 x 6 instead of d x d, and delta lies in range(J^T) by construction,
// so fp32 rounding has no self-motion component to amplify by 1/lambda: no refinement step is needed.
template <int D, bool WEIGHTED, typename SpecT>
__device__ __forceinline__ bool lm_delta_dual(const Pose<D> &P, float lam, float (&delta)[D]) {
    using K = JK<WEIGHTED, SpecT>;
    float L[6][6], invd[6], y[6];
#pragma unroll
    for (int a = 0; a < 6; ++a) {
#pragma unroll
        for (int b = 0; b <= a; ++b) { // (J J^T)_ab = sum_j J[a][j] J[b][j], lambda on the diagonal
            float acc = lam;
            bool have = (a == b);
#pragma unroll
            for (int j = 0; j < D; ++j) {
                if (K::zero(j, a) || K::zero(j, b)) continue;
                const float u = jentry<D>(P, j, a), v = jentry<D>(P, j, b);
                const bool ou = K::one(j, a), ov = K::one(j, b);
                if (ou && ov) acc = have ? add(acc, 1.f) : 1.f;
                else if (ou) acc = have ? add(acc, v) : v;
                else if (ov) acc = have ? add(acc, u) : u;
                else acc = have ? fma_(u, v, acc) : mul(u, v);
                have = true;
            }
            L[a][b] = have ? acc : 0.f;
        }
    }
    bool ok = true;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const float piv = L[k][k];
        ok = ok && (piv > 0.f);
        const float id = rsqrtf(piv);
        invd[k] = id;
#pragma unroll
        for (int i = k + 1; i < 6; ++i) L[i][k] = mul(L[i][k], id);
#pragma unroll
        for (int j = k + 1; j < 6; ++j)
#pragma unroll
            for (int i = j; i < 6; ++i) L[i][j] = fma_(-L[i][k], L[j][k], L[i][j]);
    }
    chol_solve<6>(L, invd, P.r, y);
    float asum = 0.f;
#pragma unroll
    for (int j = 0; j < D; ++j) {
        delta[j] = -colvec_k<D, WEIGHTED, SpecT>(P, j, y);
        asum = add(asum, fabsf(delta[j]));
    }
    return ok && (asum < 1e30f);
}

} // namespace lmk
