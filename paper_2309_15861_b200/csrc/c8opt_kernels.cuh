// c8opt_kernels.cuh -- device code of the photon path (sm_100a).
//
// One kernel does the whole path of SURVEY.md §8(a): per-segment preamble (a1, fp64),
// Philox draw (a2), photon generation (a3), plane projection + telescope-sphere test (a4)
// and tally / record output (a5).  Citations: PAPER.md:<line> = the paper, R<n> = a reading
// listed in DESIGN.md §2.  Nothing here is shared with oracle/ (written independently).
//
// Work decomposition: a thread block owns a *tile* of kTile emitters, an
// emitter being one (segment, process) pair.  Phase 1: thread t computes the fp64 preamble
// of emitter t and leaves an fp32 frame in shared memory.  Phase 2: the photons of the
// tile form one concatenated index space (exclusive scan of the bunch counts n_b); warp w
// walks a contiguous 1/8 of it 32 photons at a time, so every lane always has a photon
// regardless of how many photons each segment emits.  A lane keeps the frame of its
// current emitter in registers and reloads it only when its photon index crosses into the
// next emitter.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace c8 {

constexpr int kTile = 256;            // emitters per tile == threads per block
constexpr int kWarps = kTile / 32;
constexpr int kFrameStride = 36;      // floats per emitter frame in shared memory (144 B)
constexpr int kTelSmemMax = 128;      // telescopes staged (and tallied) in shared memory
constexpr int kMaxLayers = 8;

constexpr int KIND_CHER_AXIS = 0;     // Cherenkov, axis-relative projection (|d_z| large)
constexpr int KIND_FL_ISO = 1;        // fluorescence, isotropic
constexpr int KIND_CONE = 2;          // fluorescence beamed (random polar angle in a cone)
constexpr int KIND_CHER_GEN = 3;      // Cherenkov, generic projection (near-horizontal / upward track)

struct LayerD { double h_lo, a, b, c; };
struct LayerF { float h_lo, a, b, inv_c; };

struct Tally { unsigned long long hits; double sum_w; double sum_wt; };

// Everything the kernel needs, passed by value (constant bank).
struct KParams {
    // atmosphere
    int n_layers;
    LayerD layer[kMaxLayers];
    LayerF layerf[kMaxLayers];
    double eta0, rho0;
    float kappa_m;                 // 0.01 * eta0 / rho0 : metres of excess optical path per g/cm^2 (R8)
    const float *tau;              // device, [tau_nh][tau_nl] or nullptr
    int tau_nh, tau_nl;
    float tau_h0, tau_inv_dh, tau_l0, tau_inv_dl;
    // telescopes
    int n_tel;
    const float4 *telA;            // device: (cx - x_ref, cy - y_ref, cz - z_ref, R^2)
    const float *telT;             // device: column depth T(c_z) [g/cm^2]
    double x_ref, y_ref, z_ref;
    // run
    uint32_t key0, key1;
    uint32_t processes, n_procs;
    double c_ft;                   // 2 pi alpha (1/lam1 - 1/lam2) [1/m]  (R2)
    double bunch_size, fl_yield;
    float inv_lam1, dinv_lam;      // Cherenkov: 1/lam = inv_lam1 - u3 * dinv_lam (R4)
    float fl_lam1, fl_dlam;
    int beam_tel;
    double beam_x, beam_y, beam_z; // centre of the beam telescope (absolute)
    double omc;                    // 1 - cos(alpha_b) (R14)
    // work
    const float4 *seg;             // device, 3 x float4 per segment
    unsigned long long n_seg, first_id;
    // results
    Tally *tallies;                // device [n_tel]
    unsigned long long *counters;  // device [8]
    unsigned long long *cursors;   // device [n_tel]  (photon-output mode)
    float *records; const unsigned long long *tel_offset, *tel_capacity;
    unsigned long long *ids; uint32_t *counts;
};

__device__ __forceinline__ uint32_t lane_id() { return threadIdx.x & 31u; }

// ------------------------------------------------------------------------------------
// a2: Philox4x32-10 (Salmon et al., SC'11), counter (j, S_lo, S_hi, tag), key = seed (R20).
struct Rand4 { uint32_t r0, r1, r2, r3; };

__device__ __forceinline__ Rand4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned long long pa = (unsigned long long)0xD2511F53u * c0;
        const unsigned long long pb = (unsigned long long)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(pb >> 32) ^ c1 ^ k0;
        const uint32_t n2 = (uint32_t)(pa >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)pb; c3 = (uint32_t)pa; c0 = n0; c2 = n2;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return Rand4{c0, c1, c2, c3};
}

// R19: U = ((r >> 9) + 1/2) 2^-23.  one_two(r) = 1 + (r >> 9) 2^-23 in [1, 2) by mantissa stuffing;
// U = one_two(r) - kOneMinus with kOneMinus = 1 - 2^-24 (the subtraction is exact in fp32).
__device__ __forceinline__ float one_two(uint32_t r) { return __uint_as_float(0x3f800000u | (r >> 9)); }
constexpr float kOneMinus = 0.99999994f;   // 1 - 2^-24 = 0x3f7fffff
__device__ __forceinline__ float uniform01(uint32_t r) { return one_two(r) - kOneMinus; }

// ------------------------------------------------------------------------------------
// shared-memory layout of one tile
struct TileSmem {
    uint32_t prefix[kTile + 8];                 // exclusive scan of n_b; prefix[kTile] = total
    float frame[kTile * kFrameStride];          // fp32 frames, see frame slots below
    uint8_t kind[kTile];
    uint8_t invalid[kTile];
    uint32_t warp_sum[kWarps];
    float4 telA[kTelSmemMax];
    float telT[kTelSmemMax];
    uint32_t t_hits[kTelSmemMax];
    double t_sw[kTelSmemMax], t_swt[kTelSmemMax];
    unsigned long long n_upward;
};

// frame slots.  Axis-relative Cherenkov (KIND_CHER_AXIS):
//   F_NEGL   -L                      F_K0C  K0 + (1-2^-24) L,  K0 = -(z0 - z_ref)/d_z  (axis path length to the plane)
//   F_AZ..CZ v_z = CZ + cos'*AZ + sin'*BZ   (cos', sin' are of phi - pi, so AZ, BZ, P, Q carry a minus sign)
//   F_PX..QY N = cos'*P + sin'*Q  : in-plane offset direction, ground = G + (sd / v_z) N
//   F_GX,GY  where the track axis crosses the plane z_ref, relative to (x_ref, y_ref)
// Generic kinds: F_E0..2 start point relative to (x_ref, y_ref, z_ref), F_D0..2 direction, F_L,
//   F_A0..C2 (7..15): v = sth (cos' A + sin' B) + cth C.
// Hit-only slots (all kinds): F_W0 weight, F_T0 start time, F_IBC 1/(beta c), and for the axis kind
//   F_DZ, F_AX..F_CY (v_x, v_y coefficients), F_LEN.
enum {
    F_NEGL = 0, F_K0C = 1, F_AZ = 2, F_BZ = 3, F_CZ = 4, F_PX = 5, F_PY = 6, F_QX = 7, F_QY = 8, F_GX = 9, F_GY = 10,
    F_E0 = 0, F_D0 = 3, F_L = 6, F_A0 = 7, F_B0 = 10, F_C0 = 13,
    F_W0 = 16, F_T0 = 17, F_IBC = 18, F_DZ = 19, F_AX = 20, F_AY = 21, F_BX = 22, F_BY = 23, F_CX = 24, F_CY = 25,
    F_LEN = 26
};

// ------------------------------------------------------------------------------------
// a1 helpers (fp64, no FMA contraction: every operation is an explicit _rn intrinsic so the
// bunch count n_b is evaluated in the operation order DESIGN.md §4 states).
__device__ __forceinline__ double dmul(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double dadd(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double dsub(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ double ddiv(double a, double b) { return __ddiv_rn(a, b); }

__device__ __forceinline__ int layer_of(const KParams &P, double h)
{
    int i = 0;
    for (int k = 1; k < P.n_layers; ++k) if (h >= P.layer[k].h_lo) i = k;
    return i;
}

// rho(h) = -dT/dh = (b/c) exp(-h/c) [g/cm^2/m] / 100 -> g/cm^3 ; eta = eta0 rho / rho0
__device__ __forceinline__ double refractivity(const KParams &P, double h)
{
    const LayerD l = P.layer[layer_of(P, h)];
    const double dens = ddiv(dmul(ddiv(l.b, l.c), exp(ddiv(-h, l.c))), 100.0);
    return ddiv(dmul(P.eta0, dens), P.rho0);
}

// Columns 0 and 1 of M_Rod = 1 + 2 R^2 for the bisector A of (dir, -z) (R6).
// Column 2 is -dir, because M maps the downward normal onto dir.
__device__ __forceinline__ void rodrigues_columns(const double dir[3], double m0[3], double m1[3])
{
    double Ax, Ay, Az;
    if (1.0 - dir[2] < 1e-12) { Ax = 1.0; Ay = 0.0; Az = 0.0; }
    else {
        const double ax = dir[0], ay = dir[1], az = dir[2] - 1.0;
        const double n = sqrt(ax * ax + ay * ay + az * az);
        Ax = ax / n; Ay = ay / n; Az = az / n;
    }
    m0[0] = 1.0 - 2.0 * Ay * Ay - 2.0 * Az * Az; m0[1] = 2.0 * Ax * Ay;                   m0[2] = 2.0 * Ax * Az;
    m1[0] = 2.0 * Ax * Ay;                   m1[1] = 1.0 - 2.0 * Ax * Ax - 2.0 * Az * Az; m1[2] = 2.0 * Ay * Az;
}

// Preamble of emitter (segment i, process tag).  Writes the frame, returns n_b.
// *bad is set when the segment is invalid (non-finite field, gamma <= 1, L < 0, |d| off unity by > 1e-3,
// or n_b >= 2^24).
__device__ uint32_t preamble(const KParams &P, const float4 s0, const float4 s1, const float4 s2, int tag,
                             float *__restrict__ fr, uint8_t *kind_out, bool *bad)
{
    *bad = false;
    const double L = (double)s1.w, gamma = (double)s2.x, zq = (double)s2.y, dE = (double)s2.z;
    const double dx = (double)s1.x, dy = (double)s1.y, dz = (double)s1.z;
    const double dn = sqrt(dadd(dadd(dmul(dx, dx), dmul(dy, dy)), dmul(dz, dz)));
    const bool finite = isfinite(s0.x) && isfinite(s0.y) && isfinite(s0.z) && isfinite(s0.w) && isfinite(dn) &&
                        isfinite(L) && isfinite(gamma) && isfinite(zq) && isfinite(dE);
    if (!finite || !(gamma > 1.0) || !(L >= 0.0) || !(fabs(dn - 1.0) <= 1e-3)) { *bad = true; return 0; }
    const double d[3] = { ddiv(dx, dn), ddiv(dy, dn), ddiv(dz, dn) };
    const double p0[3] = { (double)s0.x, (double)s0.y, (double)s0.z };
    const double ig2 = ddiv(1.0, dmul(gamma, gamma));
    const double beta = sqrt(dsub(1.0, ig2));
    const double ibc = 1.0 / (beta * 0.299792458);        // R7: the particle moves at beta c  [ns/m]

    double mu, sin_c = 0.0, cos_c = 1.0;
    int kind;
    double axis[3];
    if (tag == 0) {
        // Frank-Tamm with the atmosphere homogeneous over the step (R3: midpoint altitude).
        const double h_mid = dadd(p0[2], dmul(dmul(0.5, L), d[2]));
        const double eta = refractivity(P, h_mid);
        const double n1 = dadd(1.0, eta);
        // q = beta^2 n^2 - 1 without cancellation; q <= 0 is the threshold Theta(beta - 1/n).
        const double q = dsub(dadd(dmul(2.0, eta), dmul(eta, eta)), dmul(dmul(n1, n1), ig2));
        if (!(q > 0.0) || !(L > 0.0)) return 0;
        const double bn2 = dmul(dmul(dsub(1.0, ig2), n1), n1);
        const double sin2 = ddiv(q, bn2);
        cos_c = 1.0 / sqrt(bn2);
        sin_c = sqrt(sin2);
        mu = dmul(dmul(dmul(dmul(P.c_ft, zq), zq), L), sin2);
        axis[0] = d[0]; axis[1] = d[1]; axis[2] = d[2];
        kind = (d[2] <= -0.1) ? KIND_CHER_AXIS : KIND_CHER_GEN;
    } else {
        // constant yield x total energy loss over the track (R13).
        mu = dmul(P.fl_yield, dE);
        if (P.beam_tel >= 0) {
            // PAPER.md:39, R15: line of sight from the segment midpoint to the telescope centre.
            const double bt[3] = { P.beam_x, P.beam_y, P.beam_z };
            double ln = 0.0;
            for (int i = 0; i < 3; ++i) { axis[i] = bt[i] - (p0[i] + 0.5 * L * d[i]); ln += axis[i] * axis[i]; }
            ln = sqrt(ln);
            for (int i = 0; i < 3; ++i) axis[i] /= ln;
            kind = KIND_CONE;
        } else {
            kind = KIND_FL_ISO;
            axis[0] = axis[1] = 0.0; axis[2] = -1.0;
        }
    }
    if (!(mu > 0.0)) return 0;
    const double nb = ceil(ddiv(mu, P.bunch_size));              // R1: deterministic bunches
    if (nb > 16777215.0) { *bad = true; return 0; }
    double w0 = ddiv(mu, nb);
    if (kind == KIND_CONE) w0 *= 0.5 * P.omc;                    // R14: Omega / 4 pi

    fr[F_W0] = (float)w0; fr[F_T0] = s0.w; fr[F_IBC] = (float)ibc; fr[F_LEN] = (float)L;
    *kind_out = (uint8_t)kind;
    const double e0[3] = { p0[0] - P.x_ref, p0[1] - P.y_ref, p0[2] - P.z_ref };
    if (kind == KIND_FL_ISO) {
        for (int i = 0; i < 3; ++i) { fr[F_E0 + i] = (float)e0[i]; fr[F_D0 + i] = (float)d[i]; }
        fr[F_L] = (float)L;
        return (uint32_t)nb;
    }
    double m0[3], m1[3];
    rodrigues_columns(axis, m0, m1);
    if (kind == KIND_CHER_AXIS) {
        // v = cos_c d + sin_c (cos phi m0 + sin phi m1); the kernel evaluates cos', sin' of phi - pi,
        // so every coefficient of cos phi / sin phi is stored negated.
        const double K0 = -e0[2] / d[2];
        fr[F_NEGL] = (float)(-L);
        fr[F_K0C] = (float)(K0 + (double)kOneMinus * L);
        fr[F_AZ] = (float)(-sin_c * m0[2]); fr[F_BZ] = (float)(-sin_c * m1[2]); fr[F_CZ] = (float)(cos_c * d[2]);
        fr[F_PX] = (float)(-sin_c * (m0[0] * d[2] - d[0] * m0[2]));
        fr[F_PY] = (float)(-sin_c * (m0[1] * d[2] - d[1] * m0[2]));
        fr[F_QX] = (float)(-sin_c * (m1[0] * d[2] - d[0] * m1[2]));
        fr[F_QY] = (float)(-sin_c * (m1[1] * d[2] - d[1] * m1[2]));
        fr[F_GX] = (float)(e0[0] + K0 * d[0]);
        fr[F_GY] = (float)(e0[1] + K0 * d[1]);
        fr[F_DZ] = (float)d[2];
        fr[F_AX] = (float)(-sin_c * m0[0]); fr[F_AY] = (float)(-sin_c * m0[1]);
        fr[F_BX] = (float)(-sin_c * m1[0]); fr[F_BY] = (float)(-sin_c * m1[1]);
        fr[F_CX] = (float)(cos_c * d[0]);   fr[F_CY] = (float)(cos_c * d[1]);
        return (uint32_t)nb;
    }
    // KIND_CONE / KIND_CHER_GEN: v = sth (cos' A + sin' B) + cth C
    const double sa = (kind == KIND_CHER_GEN) ? sin_c : 1.0, sc = (kind == KIND_CHER_GEN) ? cos_c : 1.0;
    for (int i = 0; i < 3; ++i) {
        fr[F_E0 + i] = (float)e0[i]; fr[F_D0 + i] = (float)d[i];
        fr[F_A0 + i] = (float)(-sa * m0[i]); fr[F_B0 + i] = (float)(-sa * m1[i]); fr[F_C0 + i] = (float)(sc * axis[i]);
    }
    fr[F_L] = (float)L;
    return (uint32_t)nb;
}

// ------------------------------------------------------------------------------------
// a4/a5 rare path: a photon that passed the conservative pre-test for telescope k.
//   ez    emission altitude above z_ref            (vx, vy, vz) unit direction, rv = 1 / vz
//   gx,gy crossing of the plane z_ref relative to (x_ref, y_ref)
//   s     distance of the emission point along the track, r2 the wavelength random word
template <int MODE>
__device__ __noinline__ void candidate(const KParams &P, TileSmem &sm, int k, int e, uint32_t j, unsigned long long S,
                                       int tag, uint32_t r2, float s, float ez, float vx, float vy, float vz, float rv,
                                       float gx, float gy)
{
    const float4 T = (P.n_tel <= kTelSmemMax) ? sm.telA[k] : P.telA[k];
    const float qx = gx - T.x, qy = gy - T.y, qz = -T.z;
    const float qv = fmaf(qx, vx, fmaf(qy, vy, qz * vz));
    const float b2 = fmaf(qx, qx, fmaf(qy, qy, qz * qz)) - qv * qv;       // R10: distance^2 of the centre to the ray
    const float hk = ez - T.z;                                             // emission height above the telescope plane
    const float s_pl = -hk * rv;                                           // path length to that plane (R11)
    const float s_c = (s_pl - T.z * rv) - qv;                              // closest approach along the forward ray
    // (the point (gx, gy) is on the plane z_ref at path length -ez rv = s_pl - T.z rv)
    if (!(b2 <= T.w) || !(hk > 0.0f) || !(s_c > 0.0f)) return;

    const float *fr = &sm.frame[e * kFrameStride];
    const float habs = (float)P.z_ref + ez;
    // R8: arrival time = emission time + (geometric path + integral of eta dl) / c,
    //     integral = kappa (T(c_z) - T(e_z)) / |v_z|
    int li = 0;
    for (int i = 1; i < P.n_layers; ++i) if (habs >= P.layerf[i].h_lo) li = i;
    const LayerF lf = P.layerf[li];
    const float Te = fmaf(lf.b, __expf(-habs * lf.inv_c), lf.a);
    const float Tk = (P.n_tel <= kTelSmemMax) ? sm.telT[k] : P.telT[k];
    const float excess = P.kappa_m * (Tk - Te) * fabsf(rv);
    const float t = fmaf(s, fr[F_IBC], fr[F_T0]) + (s_pl + excess) * (1.0f / 0.299792458f);
    // R4: wavelength
    const float u3 = uniform01(r2);
    const float lam = (tag == 0) ? __frcp_rn(fmaf(-u3, P.dinv_lam, P.inv_lam1)) : fmaf(u3, P.fl_dlam, P.fl_lam1);
    // R17: transmission weight exp(-tau(h, lambda) / |v_z|)
    float w = fr[F_W0];
    if (P.tau != nullptr) {
        const int nh = P.tau_nh, nl = P.tau_nl;
        float fh = (habs - P.tau_h0) * P.tau_inv_dh, fl = (lam - P.tau_l0) * P.tau_inv_dl;
        fh = fminf(fmaxf(fh, 0.0f), (float)(nh - 1)); fl = fminf(fmaxf(fl, 0.0f), (float)(nl - 1));
        int ih = min(max((int)floorf(fh), 0), max(nh - 2, 0)), il = min(max((int)floorf(fl), 0), max(nl - 2, 0));
        const float th = fh - (float)ih, tl = fl - (float)il;
        const int ih1 = (nh > 1) ? ih + 1 : ih, il1 = (nl > 1) ? il + 1 : il;
        const float t00 = __ldg(&P.tau[ih * nl + il]), t01 = __ldg(&P.tau[ih * nl + il1]);
        const float t10 = __ldg(&P.tau[ih1 * nl + il]), t11 = __ldg(&P.tau[ih1 * nl + il1]);
        const float tau = (1.0f - th) * fmaf(tl, t01 - t00, t00) + th * fmaf(tl, t11 - t10, t10);
        w *= __expf(-tau * fabsf(rv));
    }
    // a5: tally
    if (P.n_tel <= kTelSmemMax) {
        atomicAdd(&sm.t_hits[k], 1u);
        atomicAdd(&sm.t_sw[k], (double)w);
        atomicAdd(&sm.t_swt[k], (double)w * (double)t);
    } else {
        atomicAdd(&P.tallies[k].hits, 1ull);
        atomicAdd(&P.tallies[k].sum_w, (double)w);
        atomicAdd(&P.tallies[k].sum_wt, (double)w * (double)t);
    }
    if (MODE == 1) {
        const unsigned long long slot = atomicAdd(&P.cursors[k], 1ull);
        if (slot < P.tel_capacity[k]) {
            const unsigned long long at = P.tel_offset[k] + slot;
            float *rec = P.records + at * 7ull;
            // position on the plane through the telescope centre, relative to the centre (R11)
            rec[0] = fmaf(T.z * rv, vx, qx); rec[1] = fmaf(T.z * rv, vy, qy);
            rec[2] = vx; rec[3] = vy; rec[4] = t; rec[5] = lam; rec[6] = w;
            if (P.ids) P.ids[at] = (S << 25) | ((unsigned long long)tag << 24) | (unsigned long long)j;
        }
    }
}

// Conservative pre-test over all telescopes for a downward photon; calls candidate() for survivors.
// For coplanar telescopes (q_z = 0): b^2 = |q|^2 - (q.v)^2 >= |q|^2 v_z^2, so |q|^2 v_z^2 > R^2 is a miss.
template <bool COPLANAR, int MODE>
__device__ __forceinline__ void test_telescopes(const KParams &P, TileSmem &sm, const float4 *__restrict__ tel,
                                                int e, uint32_t j, unsigned long long S, int tag, uint32_t r2, float s,
                                                float ez, float vx, float vy, float vz, float rv, float gx, float gy)
{
    const float vz2 = vz * vz;
    for (int k = 0; k < P.n_tel; ++k) {
        const float4 T = tel[k];
        const float qx = gx - T.x, qy = gy - T.y;
        bool cand;
        if (COPLANAR) {
            cand = fmaf(qy, qy, qx * qx) * vz2 <= T.w;
        } else {
            const float qv = fmaf(qx, vx, fmaf(qy, vy, -T.z * vz));
            cand = fmaf(qx, qx, fmaf(qy, qy, T.z * T.z)) - qv * qv <= T.w * 1.0001f + 1e-3f;
        }
        if (cand) candidate<MODE>(P, sm, k, e, j, S, tag, r2, s, ez, vx, vy, vz, rv, gx, gy);
    }
}

// a3 + a4 for the generic kinds (isotropic / cone / generic Cherenkov).  Returns true if the photon goes upward.
template <bool COPLANAR, int MODE>
__device__ __noinline__ bool generic_photon(const KParams &P, TileSmem &sm, const float4 *__restrict__ tel, int kind,
                                            int e, uint32_t j, unsigned long long S)
{
    const float *fr = &sm.frame[e * kFrameStride];
    const int tag = (kind == KIND_CHER_GEN) ? 0 : 1;
    const Rand4 r = philox4x32_10(j, (uint32_t)S, (uint32_t)(S >> 32), (uint32_t)tag, P.key0, P.key1);
    const float s = uniform01(r.r0) * fr[F_L];
    const float ex = fmaf(s, fr[F_D0 + 0], fr[F_E0 + 0]), ey = fmaf(s, fr[F_D0 + 1], fr[F_E0 + 1]);
    const float ez = fmaf(s, fr[F_D0 + 2], fr[F_E0 + 2]);
    // sin', cos' of phi - pi = pi (2 u2 - 1); 2 u2 - 1 is exact in fp32 (R5)
    float sp, cp;
    sincospif(fmaf(2.0f, uniform01(r.r1), -1.0f), &sp, &cp);
    float vx, vy, vz;
    if (kind == KIND_FL_ISO) {
        // R16: cos(theta) = 1 - 2 u4, v = (cos phi sin th, sin phi sin th, -cos th); cos phi = -cos'
        const float u4 = uniform01(r.r3);
        const float cth = fmaf(-2.0f, u4, 1.0f), sth = 2.0f * sqrtf(u4 * (1.0f - u4));
        vx = -cp * sth; vy = -sp * sth; vz = -cth;
    } else {
        float sth = 1.0f, cth = 1.0f;
        if (kind == KIND_CONE) {                      // R14: 1 - cos(theta') uniform in [0, 1 - cos(alpha_b)]
            const float t = uniform01(r.r3) * (float)P.omc;
            cth = 1.0f - t; sth = sqrtf(t * (2.0f - t));
        }
        vx = fmaf(sth, fmaf(cp, fr[F_A0 + 0], sp * fr[F_B0 + 0]), cth * fr[F_C0 + 0]);
        vy = fmaf(sth, fmaf(cp, fr[F_A0 + 1], sp * fr[F_B0 + 1]), cth * fr[F_C0 + 1]);
        vz = fmaf(sth, fmaf(cp, fr[F_A0 + 2], sp * fr[F_B0 + 2]), cth * fr[F_C0 + 2]);
    }
    if (!(vz < 0.0f)) return true;
    const float rv = 1.0f / vz;
    const float spl = -ez * rv;
    const float gx = fmaf(spl, vx, ex), gy = fmaf(spl, vy, ey);
    test_telescopes<COPLANAR, MODE>(P, sm, tel, e, j, S, tag, r.r2, s, ez, vx, vy, vz, rv, gx, gy);
    return false;
}

// ------------------------------------------------------------------------------------
template <bool COPLANAR, int MODE>
__global__ void __launch_bounds__(kTile, 3) propagate_kernel(const __grid_constant__ KParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    TileSmem &sm = *reinterpret_cast<TileSmem *>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int segs_per_tile = kTile / (int)P.n_procs;

    // ---- stage telescopes, clear tile tallies
    const bool tel_in_smem = P.n_tel <= kTelSmemMax;
    if (tel_in_smem) {
        for (int k = tid; k < P.n_tel; k += kTile) {
            sm.telA[k] = P.telA[k]; sm.telT[k] = P.telT[k];
            sm.t_hits[k] = 0u; sm.t_sw[k] = 0.0; sm.t_swt[k] = 0.0;
        }
    }
    if (tid == 0) sm.n_upward = 0ull;
    sm.invalid[tid] = 0;
    __syncthreads();

    // ---- phase 1: preamble of emitter tid (a1)
    const int seg_local = (P.n_procs == 2) ? (tid & (kTile / 2 - 1)) : tid;
    const int tag = (P.n_procs == 2) ? (tid >> 7) : ((P.processes & 1u) ? 0 : 1);
    const unsigned long long seg_i = (unsigned long long)blockIdx.x * (unsigned)segs_per_tile + (unsigned)seg_local;
    uint32_t nb = 0;
    if (seg_i < P.n_seg) {
        const float4 *sp = P.seg + seg_i * 3ull;
        const float4 s0 = __ldg(sp), s1 = __ldg(sp + 1), s2 = __ldg(sp + 2);
        bool bad;
        nb = preamble(P, s0, s1, s2, tag, &sm.frame[tid * kFrameStride], &sm.kind[tid], &bad);
        if (bad) sm.invalid[seg_local] = 1;
        if (P.counts) {
            P.counts[seg_i * 2ull + (unsigned)tag] = nb;
            if (P.n_procs == 1) P.counts[seg_i * 2ull + (unsigned)(tag ^ 1)] = 0u;
        }
    }
    // ---- exclusive scan of nb over the tile
    uint32_t inc = nb;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint32_t v = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += v; }
    if (lane == 31) sm.warp_sum[warp] = inc;
    __syncthreads();
    uint32_t woff = 0, total = 0;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) { const uint32_t v = sm.warp_sum[w]; if (w < warp) woff += v; total += v; }
    sm.prefix[tid] = woff + inc - nb;
    if (tid < 8) sm.prefix[kTile + tid] = (tid == 0) ? total : 0xffffffffu;
    __syncthreads();

    // ---- phase 2: warp `warp` walks photons [lo, hi) of the tile's concatenated index space
    const uint32_t lo = (uint32_t)(((unsigned long long)total * (unsigned)warp) / kWarps);
    const uint32_t hi = (uint32_t)(((unsigned long long)total * (unsigned)(warp + 1)) / kWarps);
    const float4 *tel = tel_in_smem ? sm.telA : P.telA;
    const unsigned long long tile_first = P.first_id + (unsigned long long)blockIdx.x * (unsigned)segs_per_tile;
    uint32_t n_up = 0;

    if (lo < hi) {
        // emitter of this lane's first photon: the last e with prefix[e] <= g (skips empty emitters)
        int e;
        {
            const uint32_t g = min(lo + (uint32_t)lane, hi - 1u);
            int a = 0, b = kTile;                 // invariant: prefix[a] <= g < prefix[b]
            while (b - a > 1) { const int m = (a + b) >> 1; if (sm.prefix[m] <= g) a = m; else b = m; }
            e = a;
        }
        uint32_t start = sm.prefix[e], end = sm.prefix[e + 1];
        int kind = sm.kind[e];
        unsigned long long S = tile_first + (unsigned)((P.n_procs == 2) ? (e & (kTile / 2 - 1)) : e);
        float f0, f1, f2, f3, f4, f5, f6, f7, f8, f9, f10;
        {
            const float4 *fp = reinterpret_cast<const float4 *>(&sm.frame[e * kFrameStride]);
            const float4 A = fp[0], B = fp[1], C = fp[2];
            f0 = A.x; f1 = A.y; f2 = A.z; f3 = A.w; f4 = B.x; f5 = B.y; f6 = B.z; f7 = B.w; f8 = C.x; f9 = C.y; f10 = C.z;
        }
        for (uint32_t base = lo; base < hi; base += 32u) {
            const uint32_t g = base + (uint32_t)lane;
            if (g >= hi) continue;
            if (g >= end) {
                do { ++e; end = sm.prefix[e + 1]; } while (g >= end);
                start = sm.prefix[e];
                kind = sm.kind[e];
                S = tile_first + (unsigned)((P.n_procs == 2) ? (e & (kTile / 2 - 1)) : e);
                const float4 *fp = reinterpret_cast<const float4 *>(&sm.frame[e * kFrameStride]);
                const float4 A = fp[0], B = fp[1], C = fp[2];
                f0 = A.x; f1 = A.y; f2 = A.z; f3 = A.w; f4 = B.x; f5 = B.y; f6 = B.z; f7 = B.w; f8 = C.x; f9 = C.y; f10 = C.z;
            }
            const uint32_t j = g - start;
            if (kind == KIND_CHER_AXIS) {
                // a2
                const Rand4 r = philox4x32_10(j, (uint32_t)S, (uint32_t)(S >> 32), 0u, P.key0, P.key1);
                // a3: remaining axis path length to the plane, azimuth (PAPER.md:61 c_rng, R5)
                const float w1 = one_two(r.r0);
                const float sd = fmaf(w1, f0, f1);                              // K0 - u1 L
                float sp, cp;
                __sincosf(fmaf(one_two(r.r1), 6.2831853f, -9.42477760f), &sp, &cp);   // phi - pi, in [-pi, pi)
                const float vz = fmaf(cp, f2, fmaf(sp, f3, f4));
                if (!(vz < 0.0f)) { ++n_up; continue; }
                // a4: ground = G + (sd / v_z) N,  N = cos' P + sin' Q
                const float rv = __frcp_rn(vz);
                const float rho = sd * rv;
                const float gx = fmaf(rho, fmaf(cp, f5, sp * f7), f9);
                const float gy = fmaf(rho, fmaf(cp, f6, sp * f8), f10);
                const float vz2 = vz * vz;
                for (int k = 0; k < P.n_tel; ++k) {
                    const float4 T = tel[k];
                    const float qx = gx - T.x, qy = gy - T.y;
                    bool cand;
                    const float *fr = &sm.frame[e * kFrameStride];
                    if (COPLANAR) {
                        cand = fmaf(qy, qy, qx * qx) * vz2 <= T.w;
                    } else {
                        const float vx = fmaf(cp, fr[F_AX], fmaf(sp, fr[F_BX], fr[F_CX]));
                        const float vy = fmaf(cp, fr[F_AY], fmaf(sp, fr[F_BY], fr[F_CY]));
                        const float qv = fmaf(qx, vx, fmaf(qy, vy, -T.z * vz));
                        cand = fmaf(qx, qx, fmaf(qy, qy, T.z * T.z)) - qv * qv <= T.w * 1.0001f + 1e-3f;
                    }
                    if (cand) {
                        const float vx = fmaf(cp, fr[F_AX], fmaf(sp, fr[F_BX], fr[F_CX]));
                        const float vy = fmaf(cp, fr[F_AY], fmaf(sp, fr[F_BY], fr[F_CY]));
                        const float s = (w1 - kOneMinus) * fr[F_LEN];
                        const float ez = -sd * fr[F_DZ];
                        candidate<MODE>(P, sm, k, e, j, S, 0, r.r2, s, ez, vx, vy, vz, rv, gx, gy);
                    }
                }
            } else {
                if (generic_photon<COPLANAR, MODE>(P, sm, tel, kind, e, j, S)) ++n_up;
            }
        }
    }

    // ---- tile epilogue: counters and tallies
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) n_up += __shfl_xor_sync(0xffffffffu, n_up, o);
    if (lane == 0 && n_up) atomicAdd(&sm.n_upward, (unsigned long long)n_up);
    __syncthreads();
    if (tid == 0) {
        if (total) atomicAdd(&P.counters[1], (unsigned long long)total);
        if (sm.n_upward) atomicAdd(&P.counters[2], sm.n_upward);
    }
    {
        // invalid segments of this tile (each counted once)
        uint32_t nbad = (tid < segs_per_tile) ? sm.invalid[tid] : 0u;
        nbad = __reduce_add_sync(0xffffffffu, nbad);
        if (lane == 0 && nbad) atomicAdd(&P.counters[6], (unsigned long long)nbad);
    }
    if (tel_in_smem) {
        for (int k = tid; k < P.n_tel; k += kTile) {
            const uint32_t h = sm.t_hits[k];
            if (h) {
                atomicAdd(&P.tallies[k].hits, (unsigned long long)h);
                atomicAdd(&P.tallies[k].sum_w, sm.t_sw[k]);
                atomicAdd(&P.tallies[k].sum_wt, sm.t_swt[k]);
            }
        }
    }
}

}  // namespace c8
