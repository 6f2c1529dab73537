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
// next emitter.  The hot loop only decides, with a conservative pre-test, which (photon,
// telescope) pairs can be hits (~0.4 % of the photons) and pushes their 8-byte ids into a
// per-warp queue; whenever 32 are queued the warp processes them with all lanes busy:
// regenerate the photon from its counter-based random stream, exact sphere test, arrival
// time, wavelength, weight, tally / record.  Photon output with a detector that catches a
// good part of the light takes the dense loop instead (walk_dense: every candidate is
// evaluated on the spot, records staged per warp, slots reserved once per tile and round
// without a block barrier, 16-byte vector stores).  Flat photons (|v_z| < 0.05) are set
// aside and evaluated in double at the end of the tile (flat_pass).  Brute-force kernels
// (<= 8 telescopes): the preamble also finds the telescopes an emitter can reach at all; a
// trip of the pair loop whose lanes reach none only draws, orients and counts its photons.
// TEL_DISP instances: the Cherenkov launch of a request with n(lambda) (R30).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace c8 {

constexpr int kTile = 256;            // emitters per tile == threads per block
constexpr int kWarps = kTile / 32;
constexpr int kFrameStride = 36;      // floats per emitter frame in shared memory (144 B)
constexpr int kTelSmemMax = 128;      // telescopes tallied in shared memory
constexpr int kTelConstMax = 8;       // telescopes kept in the kernel-parameter constant bank
constexpr int kTelGridMin = 9;        // from this many telescopes on, the ground-plane grid replaces the brute-force pre-tests
constexpr int TEL_CONST = 0;          // brute force over <= kTelConstMax telescopes read from the constant bank
constexpr int TEL_GRID = 1;           // candidate lookup in the ground-plane grid
constexpr int TEL_GLOBAL = 2;         // brute force over telescopes in global memory (grid not buildable)
constexpr int TEL_DISP = 4;           // + TEL_DISP: the same with the wavelength-dependent refractive index (R30): the
                                      // instances the Cherenkov launch of a request with cauchy_b > 0 runs on
__host__ __device__ constexpr int tel_base(int telsrc) { return telsrc & 3; }
__host__ __device__ constexpr bool tel_disp(int telsrc) { return (telsrc & TEL_DISP) != 0; }
constexpr int kMaxLayers = 8;
constexpr int kRecWords = 7;          // floats per photon record {x, y, cos_x, cos_y, t, lambda, w}
constexpr int kBlockRecs = 64;        // photon output, dense tiles: records a warp stages per trip of the dense loop (2 per lane)
constexpr int kWarpStageWords = 2 * 2 * 64 * 7;   // floats of staging per warp: NB buffers of SUB trips x 64 records (dense loop)
#ifndef C8_FAST_BUFS
#define C8_FAST_BUFS 2
#define C8_FAST_SUB 2
#endif
constexpr int kFastBufs = C8_FAST_BUFS, kFastSub = C8_FAST_SUB;   // the fast path's split of it: buffers, trips per reservation round
constexpr int kRoundSlots = 8;        // reservation rounds in flight per tile (power of two > the buffers a warp may lag)
constexpr int kProbeDense = 32;       // candidates among the kTile sampled photons from which a tile takes the dense loop (12.5 %)
constexpr int kDenseMin = 16;         // candidates in one warp iteration from which they are evaluated on the spot
constexpr int kGenericWeight = 6;     // cost of a generic-kind photon in axis-kind photons (warp load balance)
constexpr int kCullTelMax = 128;      // culling tests the telescopes one by one up to this many, else only the array's bounding sphere
constexpr uint32_t kFlagCull = 1u;    // == C8OPT_FLAG_CULL
constexpr uint32_t kFlagRefract = 2u; // == C8OPT_FLAG_REFRACT
constexpr uint32_t kFlagCutCentre = 4u, kFlagCutTel = 8u;   // == C8OPT_FLAG_CUT_CENTRE / _TELESCOPES
constexpr float kRefractVzMin = 0.25f;   // R27: the corrections apply to photons with |v_z| >= 0.25 (zenith <= 75.5 degrees)
constexpr int MODE_TALLY = 0, MODE_OUT = 1, MODE_HIST = 2;   // == C8OPT_MODE_*
constexpr int kHistMax = 1024;        // radial bins of the ground-plane profile
constexpr int kFlatList = 96;         // flat-photon candidates a tile can defer to its double-precision pass (beyond: fp32)
constexpr int kQueue = 64;            // candidate-queue entries per warp (power of two, >= 2 * 32)
constexpr int kOutCtasPerSm = 2;       // resident CTAs per SM the brute-force photon-output kernels are compiled for (register budget)

constexpr int KIND_CHER_AXIS = 0;     // Cherenkov, axis-relative projection (|d_z| large)
constexpr int KIND_FL_ISO = 1;        // fluorescence, isotropic
constexpr int KIND_CONE = 2;          // fluorescence beamed (random polar angle in a cone)
constexpr int KIND_CHER_GEN = 3;      // Cherenkov, generic projection (near-horizontal / upward track)

struct LayerD { double h_lo, a, b, c; };
struct LayerF { float h_lo, a, b, k2; };      // T(h) = a + b 2^(-h k2), k2 = log2(e) / c

struct GridLevel { int nx, ny, base; float ox, oy, inv_cell, vzmin; };   // cell index = floor(x * inv_cell + ox)
constexpr int kGridLevels = 2;        // |v_z| >= 0.5 and >= 0.1; slot kGridLevels holds level 0 with the refraction slack (R27)

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
    const float *telEta;           // device: refractivity eta(c_z)  (C8OPT_FLAG_REFRACT)
    const double4 *telD;           // device: absolute centres in double (x, y, z, R), the angular particle cut (R29)
    double cut_cos;                // cos(cut_angle_rad)
    float4 tel_c[kTelConstMax];    // the same two tables in the constant bank when n_tel <= kTelConstMax
    float telT_c[kTelConstMax];
    float telEta_c[kTelConstMax];
    double x_ref, y_ref, z_ref;
    float z_ref_f;                 // (float)z_ref
    // ground-plane candidate grids (n_tel > kTelConstMax): cell -> up to 4 telescope indices (0xffff = none).
    // Level l serves photons with |v_z| >= grid_lvl[l].vzmin (level 0 the steep ones); n_grid_levels of them exist.
    const uint2 *grid;
    int n_grid_levels;
    GridLevel grid_lvl[kGridLevels + 1];
    // segment culling (C8OPT_FLAG_CULL): bounding sphere of the telescope array about (x_ref, y_ref, z_ref)
    uint32_t flags;
    float cull_Rb;
    // C8OPT_FLAG_REFRACT: kappa T(lowest telescope) [m] bounds |eta(e_z) (e_z - c_z) - kappa (T(c_z) - T(e_z))|, so a
    // photon's arrival point moves by at most refr_cmax sin(theta0) / cos^3(theta0); 0 without the flag
    float refr_cmax, refr_two_rmax;
    // run
    uint32_t rk0[10], rk1[10];     // Philox round keys: key + r * (0x9E3779B9, 0xBB67AE85)
    uint32_t processes, n_procs;
    int tile_segs;                 // segments per tile, <= kTile / n_procs
    int split_part;                // 0: this launch runs every requested process; 1 / 2: first / second launch of a
                                   // two-process request (Cherenkov, then fluorescence): see launch() in c8opt.cu
    double c_ft;                   // 2 pi alpha (1/lam1 - 1/lam2) [1/m]  (R2)
    double bunch_size, fl_yield;
    float inv_lam1, dinv_lam;      // Cherenkov: 1/lam = inv_lam1 - u3 * dinv_lam (R4)
    float fl_lam1, fl_dlam;
    double lam1_d, lam2_d, fl_lam1_d, fl_lam2_d;             // the same bands, and the axes of the tau table, in double:
    double tau_h0_d, tau_dh_d, tau_l0_d, tau_dl_d;           // flat photons are evaluated in double (flat_hit_f64)
    int beam_tel;
    double beam_x, beam_y, beam_z; // centre of the beam telescope, or (beam_tel == -2) of the array's sphere (absolute)
    double beam_rb;                // radius of the sphere that holds every telescope sphere (beam_tel == -2, R28)
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
    // ground-plane radial profile (MODE_HIST): bins [hist_bins] + one overflow bin, about (x_ref, y_ref) on z_ref = h_obs
    Tally *hist;
    int hist_bins;
    float hist_inv_dr, hist_wscale;        // bins per metre; 2^16 / B (fixed-point unit of the tile's weight sums)
    double hist_winv;                      // B / 2^16
    // R30 (at the end: the offsets of everything above stay as they were)
    double cauchy_b, x1_d, x2_d, c_ft0;    // n - 1 = eta (1 + b / lambda^2), b [nm^2]; 1 / lam1, 1 / lam2 [1/nm]; 2 pi alpha 1e9
    float cauchy_b_f;
};

__device__ __forceinline__ uint32_t lane_id() { return threadIdx.x & 31u; }

__device__ __forceinline__ float rcp_approx(float x)
{
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// 1/x to within 1 ulp for normal x: MUFU.RCP + one Newton step (3 instructions instead of the IEEE division's ~10)
__device__ __forceinline__ float rcp_refined(float x)
{
    const float r = rcp_approx(x);
    return fmaf(r, fmaf(-x, r, 1.0f), r);
}


// ------------------------------------------------------------------------------------
// a2: Philox4x32-10 (Salmon et al., SC'11), key = seed.  Counter (R20): fluorescence photon j of segment S draws
// the block (j, S_lo, S_hi, 1); the Cherenkov photons 2k, 2k + 1 share the block (k, S_lo, S_hi, 0).
struct Rand4 { uint32_t r0, r1, r2, r3; };

constexpr uint32_t kPhiloxM0 = 0xD2511F53u, kPhiloxM1 = 0xCD9E8D57u;

__device__ __forceinline__ void philox_round(uint32_t &c0, uint32_t &c1, uint32_t &c2, uint32_t &c3, uint32_t k0, uint32_t k1)
{
    const unsigned long long pa = (unsigned long long)kPhiloxM0 * c0;
    const unsigned long long pb = (unsigned long long)kPhiloxM1 * c2;
    const uint32_t n0 = (uint32_t)(pb >> 32) ^ c1 ^ k0;
    const uint32_t n2 = (uint32_t)(pa >> 32) ^ c3 ^ k1;
    c1 = (uint32_t)pb; c3 = (uint32_t)pa; c0 = n0; c2 = n2;
}

__device__ __forceinline__ Rand4 philox4x32_10(const KParams &P, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) philox_round(c0, c1, c2, c3, P.rk0[r], P.rk1[r]);
    return Rand4{c0, c1, c2, c3};
}

// The counter is (block index, S_lo, S_hi, tag): only word 0 changes from block to block of one emitter, so
// the S-dependent halves of rounds 1 and 2 are computed once per emitter (3 words) and each block
// does 18 instead of 20 wide multiplies.  Same function, bit for bit.
struct PhiloxEmitter { uint32_t C, D, E; };

__device__ __forceinline__ PhiloxEmitter philox_emitter(const KParams &P, unsigned long long S)
{
    const unsigned long long pb = (unsigned long long)kPhiloxM1 * (uint32_t)(S >> 32);   // round 1, c2 = S_hi
    const uint32_t A = (uint32_t)(pb >> 32) ^ (uint32_t)S ^ P.rk0[0];                    // c0 after round 1
    const uint32_t B = (uint32_t)pb;                                                     // c1 after round 1
    const unsigned long long pa = (unsigned long long)kPhiloxM0 * A;                     // round 2, c0 = A
    return PhiloxEmitter{B ^ P.rk0[1], (uint32_t)(pa >> 32) ^ P.rk1[1], (uint32_t)pa};
}

__device__ __forceinline__ Rand4 philox_photon(const KParams &P, const PhiloxEmitter &pe, uint32_t j, uint32_t tag)
{
    const unsigned long long pa = (unsigned long long)kPhiloxM0 * j;                     // round 1, c0 = j
    const uint32_t c2_1 = (uint32_t)(pa >> 32) ^ tag ^ P.rk1[0];
    const uint32_t c3_1 = (uint32_t)pa;
    const unsigned long long pb = (unsigned long long)kPhiloxM1 * c2_1;                  // round 2, c2
    uint32_t c0 = (uint32_t)(pb >> 32) ^ pe.C, c1 = (uint32_t)pb, c2 = c3_1 ^ pe.D, c3 = pe.E;
#pragma unroll
    for (int r = 2; r < 10; ++r) philox_round(c0, c1, c2, c3, P.rk0[r], P.rk1[r]);
    return Rand4{c0, c1, c2, c3};
}

// R19: U = ((r >> 9) + 1/2) 2^-23.  one_two(r) = 1 + (r >> 9) 2^-23 in [1, 2) by mantissa stuffing;
// U = one_two(r) - kOneMinus with kOneMinus = 1 - 2^-24 (the subtraction is exact in fp32).
__device__ __forceinline__ float one_two(uint32_t r) { return __uint_as_float(0x3f800000u | (r >> 9)); }
constexpr float kOneMinus = 0.99999994f;   // 1 - 2^-24 = 0x3f7fffff
__device__ __forceinline__ float uniform01(uint32_t r) { return one_two(r) - kOneMinus; }

// R20: one Philox block, counter (j >> 1, S, tag 0), serves the Cherenkov photons 2k and 2k + 1: the even one takes the
// words (r0, r1), the odd one (r2, r3).  Position and azimuth use the upper 23 bits of the photon's two words (R19); the
// wavelength uniform is built from the 9 + 9 lower bits they leave over: ((a & 511) 2^9 + (b & 511) + 1/2) 2^-18.
__device__ __forceinline__ Rand4 cherenkov_words(const Rand4 blk, uint32_t j)
{
    return (j & 1u) ? Rand4{blk.r2, blk.r3, 0u, 0u} : Rand4{blk.r0, blk.r1, 0u, 0u};
}
__device__ __forceinline__ float cherenkov_u3(uint32_t a, uint32_t b)
{
    return fmaf((float)(((a & 511u) << 9) | (b & 511u)), 3.814697265625e-06f, 1.9073486328125e-06f);   // exact: 18 bits
}

// ------------------------------------------------------------------------------------
// shared-memory layout of one tile
struct __align__(16) TileSmem {
    uint32_t prefix[kTile + 8];                 // exclusive scan of n_b; prefix[kTile] = total
    float frame[kTile * kFrameStride];          // fp32 frames, see frame slots below
    uint8_t kind[kTile];
    uint8_t tmask[kTile];                       // constant-bank telescopes the emitter can reach (reach_mask)
    uint8_t invalid[kTile];
    uint32_t warp_sum[kWarps], warp_pad[kWarps];
    uint8_t odd[kTile + 8];                     // 1 = the emitter's count is odd: its last slot of the index space is empty
    unsigned long long warp_wsum[kWarps];
    uint32_t bound[kWarps + 1];                 // photon ranges of the warps
    uint32_t t_hits[kTelSmemMax];
    double t_sw[kTelSmemMax], t_swt[kTelSmemMax];
    unsigned long long n_upward, n_culled;
    uint2 queue[kWarps][kQueue];                // per-warp ring of candidate (photon, telescope) pairs
    uint32_t wide_list[kWarps][64];             // photons waiting for the wide test: j | e << 24
    uint32_t wide_count[kWarps];
    uint2 flat_list[kFlatList];                 // (photon, telescope) pairs of flat photons, evaluated in double at the end of the tile
    uint32_t flat_count, flat_pad[3];
    // per-thread tally accumulators (flushed into t_* when the telescope changes and at the end of the tile)
    double acc_w[kTile], acc_wt[kTile];
    uint32_t acc_n[kTile];
    int acc_k[kTile];
};

// Photon-output kernels only (follows TileSmem in dynamic shared memory).  Dense tiles (most photons hit one telescope:
// c5g) stage the records of a trip per warp and reserve their slots once per (tile, trip): same-address atomics
// serialise in L2 (~1 per clock), so the cursor of a telescope must not be bumped once per warp and trip.  The
// reservation is a split arrive / wait without a block barrier (walk_dense): a warp adds its record count to agg[r & 3]
// (bits 8.. = records so far = the warp's offset in the round, bits 0..7 = warps arrived); the last of the kWarps
// arrivals bumps the cursor by the round's total, publishes the base in rbase[r & 7] and arrives at the mbarrier
// rbar[r & 7]; a warp picks the base up after it has staged the next block (mbarrier try_wait: the hardware parks the
// warp, no polling instructions) and copies its block out with 16-byte vector stores.
struct OutSmem {
    unsigned long long rbase[kRoundSlots];       // first record slot of round r in the dense telescope's region
    unsigned long long rbar[kRoundSlots];        // mbarrier (1 arrival): phase r / kRoundSlots completes when rbase[r % kRoundSlots] is round r's
    uint32_t agg[kRoundSlots];                   // see above
    uint32_t probe[kTelConstMax];                // candidates per telescope among the sampled photons (probe_density)
    // NB buffers per warp: block r is staged in buffer r % NB while the blocks r - 1 .. r - NB + 1 wait for their slots.
    // The general path uses two buffers of kBlockRecs records and keeps their ids (if the caller wants them) behind them.
    __align__(16) float stage[kWarps][kWarpStageWords];
};
static_assert(kFastBufs * kFastSub * kBlockRecs * kRecWords <= kWarpStageWords, "fast-path staging fits");
static_assert(2 * (kBlockRecs * kRecWords + 2 * kBlockRecs) <= kWarpStageWords, "general-path staging with ids fits");

__device__ __forceinline__ OutSmem &out_smem(TileSmem &sm)
{
    static_assert(sizeof(TileSmem) % 16 == 0, "OutSmem must stay 16-byte aligned");
    return *reinterpret_cast<OutSmem *>(&sm + 1);
}

// Ground-histogram kernel only (follows TileSmem in dynamic shared memory): the tile's private radial histogram.
// Shared memory has native atomics for 32-bit integers only (an fp32 or 64-bit add is a compare-and-swap loop, ~35
// instructions under contention), so the tile's sums are kept in fixed point: w in units of B 2^-16 (w <= B, the
// bunch size), t in units of 1/64 ns, each sum as a (lo, hi) pair of u32 with the carry propagated by hand.  The
// roundings are unbiased: 8e-6 relative per bunch weight, 8 ps per arrival time.
struct HistSmem {
    uint32_t n[kHistMax];
    uint32_t sw_lo[kHistMax], sw_hi[kHistMax];
    uint32_t swt_lo[kHistMax], swt_hi[kHistMax];     // two's-complement 64-bit sum of q_w * q_t
    uint32_t overflow;
};

__device__ __forceinline__ HistSmem &hist_smem(TileSmem &sm) { return *reinterpret_cast<HistSmem *>(&sm + 1); }

// frame slots.  Axis-relative Cherenkov (KIND_CHER_AXIS):
//   F_NEGL   -L                      F_K0C  K0 + (1-2^-24) L,  K0 = -(z0 - z_ref)/d_z  (axis path length to the plane)
//   F_AZ..CZ v_z = CZ + cos'*AZ + sin'*BZ   (cos', sin' are of phi - pi, so AZ, BZ, P, Q carry a minus sign)
//   F_PX..QY N = cos'*P + sin'*Q  : in-plane offset direction, ground = G + (sd / v_z) N
//   F_GX,GY  where the track axis crosses the plane z_ref, relative to (x_ref, y_ref)
// Generic kinds: F_E0..2 start point relative to (x_ref, y_ref, z_ref), F_D0..2 direction, F_L,
//   F_A0..C2 (7..15): v = sth (cos' A + sin' B) + cth C.
// Hit-only slots (all kinds): F_W0 weight, F_T0 start time, F_IBC 1/(beta c), and for the axis kind
//   F_DZ, F_AX..F_CY (v_x, v_y coefficients), F_LEN; F_LAYER = bits of the int index of the atmosphere layer that
//   holds the lower end of the segment, F_HNEXT = lower bound of the next layer if the segment reaches into it (else
//   +inf), F_LAYER = -1 if it spans more than two layers; F_OMC = 1 - cos(half-angle) of a beamed emitter's cone.
// Fluorescence kinds: the polar window outside of which no photon of the emitter can reach the array (polar_cull):
//   F_VZLO, F_VZHI bound v_z of an isotropic photon, F_TMAX bounds 1 - cos(theta') of a beamed one.
enum {
    F_NEGL = 0, F_K0C = 1, F_AZ = 2, F_BZ = 3, F_CZ = 4, F_PX = 5, F_PY = 6, F_QX = 7, F_QY = 8, F_GX = 9, F_GY = 10,
    F_E0 = 0, F_D0 = 3, F_L = 6, F_A0 = 7, F_B0 = 10, F_C0 = 13,
    F_W0 = 16, F_T0 = 17, F_IBC = 18, F_DZ = 19, F_AX = 20, F_AY = 21, F_BX = 22, F_BY = 23, F_CX = 24, F_CY = 25,
    F_LEN = 26, F_LAYER = 27, F_OMC = 28, F_HNEXT = 29, F_VZLO = 30, F_VZHI = 31, F_TMAX = 32,
    // R30 (Cherenkov emitters of the TEL_GLOBAL_DISP instances, generic kind; slots of the axis kind): eta(h_mid) and
    // 1 / gamma^2, each as fp32 head + tail, and 1 / <sin^2 theta_c>
    F_DETA = 19, F_DIG2 = 20, F_DINVM = 21, F_DETA_LO = 22, F_DIG2_LO = 23
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

// Segment culling, exact and conservative.  A photon leaves the track at angle theta_c to d, so it can
// reach the sphere (c, R) from the emission point e only if |angle(d, c - e) - theta_c| <= asin(R / |c - e|).  Over
// the segment (midpoint m, half length hl) the direction to c swings by at most asin(hl / D) and |c - e| >= D =
// |c - m| - hl.  With a = (R + 1 cm) / D, b = hl / D and sin(asin a + asin b) <= a + b, the sphere is out of reach if
// cos(psi - theta_c) <= 0 or |sin(psi - theta_c)| > a + b + 2e-5 (the slack covers the fp32 photon directions and
// this test's own rounding).  Returns true when the sphere CAN be hit (or the test cannot tell).
__device__ __forceinline__ bool cone_reaches(float ux, float uy, float uz, float R, float dx, float dy, float dz, float hl,
                                             float sin_c, float cos_c)
{
    // MUFU-grade rsqrt / reciprocal (2 ulp) are ample against the 2e-5 slack
    const float uu = fmaf(ux, ux, fmaf(uy, uy, uz * uz));
    const float inv = rsqrtf(uu), D = fmaf(uu, inv, -hl);
    if (!(D > R + 0.01f)) return true;
    const float sA = fmaf(R + 0.01f + hl, rcp_approx(D), 2e-5f);
    if (!(sA < 1.0f)) return true;
    const float cpsi = fmaf(dx, ux, fmaf(dy, uy, dz * uz)) * inv;
    const float cx = fmaf(dy, uz, -(dz * uy)), cy = fmaf(dz, ux, -(dx * uz)), cz = fmaf(dx, uy, -(dy * ux));
    const float cc = fmaf(cx, cx, fmaf(cy, cy, cz * cz));
    const float spsi = cc * rsqrtf(fmaxf(cc, 1e-30f)) * inv;
    const float s = fmaf(spsi, cos_c, -(cpsi * sin_c)), c = fmaf(cpsi, cos_c, spsi * sin_c);
    return c > 0.0f && fabsf(s) <= sA;
}

// true = no photon of this Cherenkov emitter can hit any telescope.  m = segment midpoint relative to the reference
// point; first the array's bounding sphere, then (small arrays) every telescope.
__device__ __noinline__ bool cull_emitter(const KParams &P, float mx, float my, float mz, float dx, float dy, float dz, float hl,
                                          float sin_c, float cos_c)
{
    // With the refraction corrections a photon lands up to refr_cmax sin / cos^3 off its straight line (R27).  The
    // photons of this emitter lie within theta_c of d, so |v_z| >= |d_z| cos_c - sqrt(1 - d_z^2) sin_c; the corrections
    // stop at |v_z| = kRefractVzMin, where the reach is 62 refr_cmax.
    float grow = 0.0f;
    if (P.flags & kFlagRefract) {
        const float vzm = fmaxf(fmaf(fabsf(dz), cos_c, -sqrtf(fmaxf(fmaf(-dz, dz, 1.0f), 0.0f)) * sin_c) - 1e-3f, kRefractVzMin);
        grow = 1.02f * P.refr_cmax * sqrtf(fmaxf(fmaf(-vzm, vzm, 1.0f), 0.0f)) / (vzm * vzm * vzm) + 0.01f;
    }
    if (!cone_reaches(-mx, -my, -mz, P.cull_Rb + grow, dx, dy, dz, hl, sin_c, cos_c)) return true;
    if (P.n_tel > kCullTelMax) return false;
    for (int k = 0; k < P.n_tel; ++k) {
        const float4 T = __ldg(&P.telA[k]);
        const float R = T.w * rsqrtf(fmaxf(T.w, 1e-30f)) + grow;
        if (cone_reaches(T.x - mx, T.y - my, T.z - mz, R, dx, dy, dz, hl, sin_c, cos_c)) return false;
    }
    return true;
}

// Which of the <= kTelConstMax constant-bank telescopes can a photon of this Cherenkov emitter reach at all?  The culling
// test, telescope by telescope (bit k = telescope k); 0xff when the question does not apply (ground histogram).  The
// pair loop skips the pre-tests of the telescopes that no lane of the warp can reach (walk_pairs).
__device__ __noinline__ uint32_t reach_mask(const KParams &P, float mx, float my, float mz, float dx, float dy, float dz, float hl,
                                            float sin_c, float cos_c)
{
    if (P.hist != nullptr || P.n_tel > kTelConstMax) return 0xffu;
    float grow = 0.0f;
    if (P.flags & kFlagRefract) {
        const float vzm = fmaxf(fmaf(fabsf(dz), cos_c, -sqrtf(fmaxf(fmaf(-dz, dz, 1.0f), 0.0f)) * sin_c) - 1e-3f, kRefractVzMin);
        grow = 1.02f * P.refr_cmax * sqrtf(fmaxf(fmaf(-vzm, vzm, 1.0f), 0.0f)) / (vzm * vzm * vzm) + 0.01f;
    }
    if (!cone_reaches(-mx, -my, -mz, P.cull_Rb + grow, dx, dy, dz, hl, sin_c, cos_c)) return 0u;
    uint32_t m = 0u;
    for (int k = 0; k < P.n_tel; ++k) {
        const float4 T = P.tel_c[k];
        const float R = T.w * rsqrtf(fmaxf(T.w, 1e-30f)) + grow;
        if (cone_reaches(T.x - mx, T.y - my, T.z - mz, R, dx, dy, dz, hl, sin_c, cos_c)) m |= 1u << k;
    }
    return m;
}

// The paper's angular particle cut (R29): true = the Cherenkov segment is not handled, because its
// direction d is more than the cut angle off the vector from its midpoint to the experiment centre (or, kFlagCutTel,
// to every telescope centre).  angle > cut is decided as d.u < cos(cut) |u|, in double, explicit round-to-nearest
// operations in the oracle's order, so that both sides cut the same segments.
__device__ __noinline__ bool particle_cut(const KParams &P, double p0x, double p0y, double p0z, double dx, double dy, double dz, double L)
{
    const double p0[3] = { p0x, p0y, p0z }, d[3] = { dx, dy, dz };
    const int n = (P.flags & kFlagCutTel) ? P.n_tel : 1;
    const double hl = dmul(0.5, L);
    for (int k = 0; k < n; ++k) {
        double c[3] = { P.x_ref, P.y_ref, P.z_ref };
        if (P.flags & kFlagCutTel) { const double4 T = P.telD[k]; c[0] = T.x; c[1] = T.y; c[2] = T.z; }
        double u[3];
        for (int i = 0; i < 3; ++i) u[i] = dsub(c[i], dadd(p0[i], dmul(hl, d[i])));
        const double dot = dadd(dadd(dmul(d[0], u[0]), dmul(d[1], u[1])), dmul(d[2], u[2]));
        const double norm = sqrt(dadd(dadd(dmul(u[0], u[0]), dmul(u[1], u[1])), dmul(u[2], u[2])));
        if (!(dot < dmul(P.cut_cos, norm))) return false;
    }
    return true;
}

// What the preamble knows about an emitter, in double: for the photons that fp32 cannot carry (flat_hit_f64).
struct FrameD { double p0[3], d[3], L, t0, ibc, w0, sin_c, cos_c, omc, axis[3]; int kind; };
struct FrameDisp { double d_eta, d_beta2, d_mean; };     // R30: refractivity at the midpoint, beta^2, band average of sin^2

// Preamble of emitter (segment i, process tag).  Writes the frame, returns n_b.
// *bad is set when the segment is invalid: 1 = non-finite field, gamma <= 1, L < 0 or |d| off unity by > 1e-3 (the
// same for both processes), 2 = n_b >= 2^24 for this process.
// DISP: the Cherenkov yield and angle with n(lambda) (R30).
template <bool WITH_D = false, bool WITH_MASK = false, bool DISP = false>
__device__ uint32_t preamble(const KParams &P, const float4 s0, const float4 s1, const float4 s2, int tag,
                             float *__restrict__ fr, uint8_t *kind_out, int *bad, bool *culled, FrameD *fd = nullptr,
                             uint8_t *tmask_out = nullptr, FrameDisp *fdisp = nullptr)
{
    if constexpr (WITH_MASK) *tmask_out = 0xffu;
    *bad = 0;
    *culled = false;
    const double L = (double)s1.w, gamma = (double)s2.x, zq = (double)s2.y, dE = (double)s2.z;
    const double dx = (double)s1.x, dy = (double)s1.y, dz = (double)s1.z;
    const double dn = sqrt(dadd(dadd(dmul(dx, dx), dmul(dy, dy)), dmul(dz, dz)));
    const bool finite = isfinite(s0.x) && isfinite(s0.y) && isfinite(s0.z) && isfinite(s0.w) && isfinite(dn) &&
                        isfinite(L) && isfinite(gamma) && isfinite(zq) && isfinite(dE);
    if (!finite || !(gamma > 1.0) || !(L >= 0.0) || !(fabs(dn - 1.0) <= 1e-3)) { *bad = 1; return 0; }
    const double d[3] = { ddiv(dx, dn), ddiv(dy, dn), ddiv(dz, dn) };
    const double p0[3] = { (double)s0.x, (double)s0.y, (double)s0.z };
    const double ig2 = ddiv(1.0, dmul(gamma, gamma));
    const double beta = sqrt(dsub(1.0, ig2));
    const double ibc = 1.0 / (beta * 0.299792458);        // R7: the particle moves at beta c  [ns/m]

    double mu, sin_c = 0.0, cos_c = 1.0, omc_e = P.omc;      // omc_e = 1 - cos(alpha) of this emitter's cone
    double d_eta = 0.0, d_beta2 = 1.0, d_mean = 1.0;         // R30: refractivity at the midpoint, beta^2, band average of sin^2
    constexpr bool disp = DISP;
    int kind;
    double axis[3];
    if (tag == 0) {
        // Frank-Tamm with the atmosphere homogeneous over the step (R3: midpoint altitude).
        const double h_mid = dadd(p0[2], dmul(dmul(0.5, L), d[2]));
        const double eta = refractivity(P, h_mid);
        axis[0] = d[0]; axis[1] = d[1]; axis[2] = d[2];
        if (disp) {
            // R30 (PAPER.md:45 with n(lambda)): N = 2 pi alpha z^2 L int sin^2 theta_c(x) Theta dx over x = 1 / lambda,
            // n(x) - 1 = eta (1 + b x^2), composite Simpson with 16 intervals; the oracle's operation order (feeds n_b).
            // Every photon then leaves at the angle of its own wavelength (photon_from_rand): generic projection.
            if (!(L > 0.0)) return 0;
            d_eta = eta; d_beta2 = dsub(1.0, ig2);
            const double h = ddiv(dsub(P.x1_d, P.x2_d), 16.0);
            double ends = 0.0, odd = 0.0, even = 0.0;
            for (int k = 0; k <= 16; ++k) {
                const double x = dadd(P.x2_d, dmul((double)k, h));
                const double n = dadd(1.0, dmul(eta, dadd(1.0, dmul(dmul(P.cauchy_b, x), x))));
                double f = dsub(1.0, ddiv(1.0, dmul(dmul(d_beta2, n), n)));
                if (!(f > 0.0)) f = 0.0;
                if (k == 0 || k == 16) ends = dadd(ends, f); else if (k & 1) odd = dadd(odd, f); else even = dadd(even, f);
            }
            const double S = dmul(ddiv(h, 3.0), dadd(dadd(ends, dmul(4.0, odd)), dmul(2.0, even)));
            if (!(S > 0.0)) return 0;
            mu = dmul(dmul(dmul(dmul(P.c_ft0, zq), zq), L), S);
            d_mean = ddiv(S, dsub(P.x1_d, P.x2_d));
            kind = KIND_CHER_GEN;
        } else {
            const double n1 = dadd(1.0, eta);
            // q = beta^2 n^2 - 1 without cancellation; q <= 0 is the threshold Theta(beta - 1/n).
            const double q = dsub(dadd(dmul(2.0, eta), dmul(eta, eta)), dmul(dmul(n1, n1), ig2));
            if (!(q > 0.0) || !(L > 0.0)) return 0;
            const double bn2 = dmul(dmul(dsub(1.0, ig2), n1), n1);
            const double sin2 = ddiv(q, bn2);
            cos_c = 1.0 / sqrt(bn2);
            sin_c = sqrt(sin2);
            mu = dmul(dmul(dmul(dmul(P.c_ft, zq), zq), L), sin2);
            kind = (d[2] <= -0.1) ? KIND_CHER_AXIS : KIND_CHER_GEN;
        }
    } else {
        // constant yield x total energy loss over the track (R13).
        mu = dmul(P.fl_yield, dE);
        if (P.beam_tel == -2) {
            // PAPER.md:39, R28: one emission cone around the sphere (beam_x/y/z, beam_rb) that holds every telescope,
            // sin(alpha) = (R_b + L/2) / D from the segment midpoint, and the NUMBER of photons scaled by
            // Omega / 4 pi = (1 - cos alpha) / 2.  Operation order as in the oracle (feeds n_b).  Inside the array:
            // isotropic, unscaled.
            const double bt[3] = { P.beam_x, P.beam_y, P.beam_z };
            for (int i = 0; i < 3; ++i) axis[i] = dsub(bt[i], dadd(p0[i], dmul(dmul(0.5, L), d[i])));
            const double D = sqrt(dadd(dadd(dmul(axis[0], axis[0]), dmul(axis[1], axis[1])), dmul(axis[2], axis[2])));
            const double sa = ddiv(dadd(P.beam_rb, dmul(0.5, L)), D);
            if (sa < 1.0) {
                kind = KIND_CONE;
                for (int i = 0; i < 3; ++i) axis[i] = ddiv(axis[i], D);
                const double ca = sqrt(dsub(1.0, dmul(sa, sa)));
                omc_e = ddiv(dmul(sa, sa), dadd(1.0, ca));
                mu = dmul(mu, dmul(0.5, omc_e));
            } else {
                kind = KIND_FL_ISO;
                axis[0] = axis[1] = 0.0; axis[2] = -1.0;
            }
        } else if (P.beam_tel >= 0) {
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
    if (nb > 16777215.0) { *bad = 2; return 0; }
    double w0 = ddiv(mu, nb);
    if (kind == KIND_CONE && P.beam_tel >= 0) w0 *= 0.5 * P.omc;  // R14 (weight form): Omega / 4 pi
    if ((P.flags & (kFlagCutCentre | kFlagCutTel)) && tag == 0 && particle_cut(P, p0[0], p0[1], p0[2], d[0], d[1], d[2], L)) {
        *culled = true;
        return (uint32_t)nb;
    }
    if (WITH_MASK && !DISP && tag == 0 && P.n_tel <= kTelConstMax) {        // (R30: no single cone, the mask stays full)
        // small arrays: the telescopes this emitter can reach at all; none = culled (C8OPT_FLAG_CULL)
        const double hl = 0.5 * L;
        const uint32_t tm = reach_mask(P, (float)(p0[0] + hl * d[0] - P.x_ref), (float)(p0[1] + hl * d[1] - P.y_ref), (float)(p0[2] + hl * d[2] - P.z_ref),
                                       (float)d[0], (float)d[1], (float)d[2], (float)hl, (float)sin_c, (float)cos_c);
        *tmask_out = (uint8_t)tm;
        if ((P.flags & kFlagCull) && tm == 0u) {
            *culled = true;
            return (uint32_t)nb;
        }
    } else if ((P.flags & kFlagCull) && tag == 0) {
        const double hl = 0.5 * L;
        if (cull_emitter(P, (float)(p0[0] + hl * d[0] - P.x_ref), (float)(p0[1] + hl * d[1] - P.y_ref), (float)(p0[2] + hl * d[2] - P.z_ref),
                         (float)d[0], (float)d[1], (float)d[2], (float)hl, (float)sin_c, (float)cos_c)) {
            *culled = true;
            return (uint32_t)nb;
        }
    }

    if constexpr (WITH_D) {
        for (int i = 0; i < 3; ++i) { fd->p0[i] = p0[i]; fd->d[i] = d[i]; fd->axis[i] = axis[i]; }
        fd->L = L; fd->t0 = (double)s0.w; fd->ibc = ibc; fd->w0 = w0; fd->sin_c = sin_c; fd->cos_c = cos_c; fd->omc = omc_e; fd->kind = kind;
        if constexpr (DISP) { fdisp->d_eta = d_eta; fdisp->d_beta2 = d_beta2; fdisp->d_mean = d_mean; }
    }
    fr[F_W0] = (float)w0; fr[F_T0] = s0.w; fr[F_IBC] = (float)ibc; fr[F_LEN] = (float)L; fr[F_OMC] = (float)omc_e;
    {
        // layer of both ends in fp32 altitudes as the photon loop sees them (1 m of margin against rounding)
        const float za = (float)p0[2], zb = (float)(p0[2] + L * d[2]);
        const float zlo = fminf(za, zb) - 1.0f, zhi = fmaxf(za, zb) + 1.0f;
        int la = 0, lb = 0;
        for (int i = 1; i < P.n_layers; ++i) { if (zlo >= P.layerf[i].h_lo) la = i; if (zhi >= P.layerf[i].h_lo) lb = i; }
        fr[F_LAYER] = __int_as_float(lb - la <= 1 ? la : -1);
        fr[F_HNEXT] = (lb == la + 1) ? P.layerf[lb].h_lo : __int_as_float(0x7f800000);
    }
    *kind_out = (uint8_t)kind;
    const double e0[3] = { p0[0] - P.x_ref, p0[1] - P.y_ref, p0[2] - P.z_ref };
    if (kind == KIND_FL_ISO || kind == KIND_CONE) {
        // Exact cull per photon ("it is vital that the above method must be very fast"): a photon can hit a
        // telescope only if it passes within R_b of the array centre c, i.e. only if its direction is within
        // A = asin(R_b / D) + asin((L/2) / D) of the line from the segment midpoint to c (D = |c - m| - L/2).  For an
        // isotropic photon that bounds v_z = -cos(theta), which the polar uniform alone gives, to a window; for a
        // beamed one it bounds the polar angle about the cone axis.  Photons outside are dropped before their
        // direction is built (polar_cull); the ground histogram takes every photon.
        // (fp32 is ample: the window carries 2e-5 rad of slack against 1e-6 of rounding)
        float vz_lo = -1.0f, vz_hi = 1.0f, t_max = __int_as_float(0x7f800000);
        if (P.hist == nullptr) {
            const float hl = (float)(0.5 * L);
            const float ux = -(float)(e0[0] + 0.5 * L * d[0]), uy = -(float)(e0[1] + 0.5 * L * d[1]), uz = -(float)(e0[2] + 0.5 * L * d[2]);
            const float Dm = sqrtf(fmaf(ux, ux, fmaf(uy, uy, uz * uz))), D = Dm - hl;
            const float Rb = P.cull_Rb * 1.00001f + ((P.flags & kFlagRefract) ? 62.5f * P.refr_cmax : 0.0f) + 0.02f;
            if (D > Rb * 1.0001f) {
                const float A = asinf(Rb / D) + asinf(fminf(1.0f, hl / D)) + 2e-5f;
                if (kind == KIND_FL_ISO) {
                    const float thu = acosf(fminf(1.0f, fmaxf(-1.0f, uz / Dm)));
                    vz_lo = cosf(fminf(3.14159265f, thu + A)) - 1e-5f;
                    vz_hi = cosf(fmaxf(0.0f, thu - A)) + 1e-5f;
                } else {
                    const float ca = ((float)axis[0] * ux + (float)axis[1] * uy + (float)axis[2] * uz) / Dm;
                    const float th_max = acosf(fminf(1.0f, fmaxf(-1.0f, ca))) + A + 6e-4f;      // (acos near 1 loses digits: 1e-7 in its argument is 4.5e-4 rad)
                    const float alpha_b = acosf(fmaxf(-1.0f, 1.0f - (float)omc_e));
                    // only when the whole cone points below the horizon: a dropped photon is then known to go down
                    if (acosf(fminf(1.0f, fmaxf(-1.0f, -(float)axis[2]))) + alpha_b < 1.5697f && th_max < 3.1415f)
                    { const float sh = sinf(0.5f * th_max); t_max = 2.0f * sh * sh * 1.0001f + 1e-12f; }   // 1 - cos, without cancellation
                }
            }
        }
        fr[F_VZLO] = vz_lo; fr[F_VZHI] = vz_hi; fr[F_TMAX] = t_max;
    }
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
    // (R30: sin / cos of the Cherenkov angle are the photon's own, so the columns stay unscaled as for the cone)
    const bool scaled = (kind == KIND_CHER_GEN) && !disp;
    const double sa = scaled ? sin_c : 1.0, sc = scaled ? cos_c : 1.0;
    for (int i = 0; i < 3; ++i) {
        fr[F_E0 + i] = (float)e0[i]; fr[F_D0 + i] = (float)d[i];
        fr[F_A0 + i] = (float)(-sa * m0[i]); fr[F_B0 + i] = (float)(-sa * m1[i]); fr[F_C0 + i] = (float)(sc * axis[i]);
    }
    fr[F_L] = (float)L;
    if constexpr (DISP) {
        if (kind == KIND_CHER_GEN) {
            fr[F_DETA] = (float)d_eta; fr[F_DETA_LO] = (float)(d_eta - (double)(float)d_eta);
            fr[F_DIG2] = (float)ig2; fr[F_DIG2_LO] = (float)(ig2 - (double)(float)ig2);
            fr[F_DINVM] = (float)(1.0 / d_mean);
        }
    }
    return (uint32_t)nb;
}

// Is the segment invalid for the Cherenkov process?  (rare path of the second launch of a two-process request)
__device__ __noinline__ int cherenkov_preamble_status(const KParams &P, const float4 s0, const float4 s1, const float4 s2, float *scratch_frame)
{
    int bad;
    bool culled;
    uint8_t kind;
    preamble(P, s0, s1, s2, 0, scratch_frame, &kind, &bad, &culled);
    return bad;
}
// the same with n(lambda) (R30: another yield, so another bunch count)
__device__ __noinline__ int cherenkov_preamble_status_disp(const KParams &P, const float4 s0, const float4 s1, const float4 s2, float *scratch_frame)
{
    int bad;
    bool culled;
    uint8_t kind;
    preamble<false, false, true>(P, s0, s1, s2, 0, scratch_frame, &kind, &bad, &culled);
    return bad;
}

// ------------------------------------------------------------------------------------
template <int TELSRC> __device__ __forceinline__ float4 tel_at(const KParams &P, int k)
{
    if (tel_base(TELSRC) == TEL_CONST) return P.tel_c[k];
    return __ldg(&P.telA[k]);
}
template <int TELSRC> __device__ __forceinline__ float telT_at(const KParams &P, int k)
{
    if (tel_base(TELSRC) == TEL_CONST) return P.telT_c[k];
    return __ldg(&P.telT[k]);
}
template <int TELSRC> __device__ __forceinline__ float telEta_at(const KParams &P, int k)
{
    if (tel_base(TELSRC) == TEL_CONST) return P.telEta_c[k];
    return __ldg(&P.telEta[k]);
}

// sin(pi x), cos(pi x) for x in [-1, 1] to ~1e-7 absolute: quadrant reduction to |r| <= 1/4 (exact in fp32) and
// Taylor polynomials in pi r (next terms < 3e-9).  About a third of sincospif's instructions, which also serves
// arguments outside [-1, 1] and special values.
__device__ __forceinline__ void sincospi_unit(float x, float *s, float *c)
{
    const float q = rintf(x + x);
    const float r = fmaf(-0.5f, q, x), r2 = r * r;
    const float sn = r * fmaf(r2, fmaf(r2, fmaf(r2, fmaf(r2, 0.0821458866f, -0.599264529f), 2.55016404f), -5.16771278f), 3.14159265f);
    const float cs = fmaf(r2, fmaf(r2, fmaf(r2, fmaf(r2, fmaf(r2, -0.0258068913f, 0.235330630f), -1.33526277f), 4.05871213f), -4.93480220f), 1.0f);
    const int qi = (int)q;
    const float a = (qi & 1) ? cs : sn, b = (qi & 1) ? sn : cs;        // odd quadrant: sin <- cos, cos <- -sin
    *s = (qi & 2) ? -a : a;
    *c = ((qi + 1) & 2) ? -b : b;
}

// A photon ready for the exact test: emission point e relative to (x_ref, y_ref, z_ref) or, for the
// axis kind, the crossing (gx, gy) of the plane z_ref; unit direction v; s = distance along the track.
struct Photon { float ex, ey, ez, gx, gy, vx, vy, vz, s, u3, rva; int tag; bool axis; };   // u3 = the wavelength uniform; rva = MUFU.RCP(v_z), axis kind

// a3 for a photon of emitter e, any kind, from its four random words.
// DISP (R30): a Cherenkov photon of the generic kind leaves at the angle of its own wavelength; ph.rva then carries its
// weight factor sin^2 theta_c(lambda) / <sin^2 theta_c>, 0 = below the threshold at this wavelength (no photon).
template <bool DISP = false>
__device__ __forceinline__ Photon photon_from_rand(const KParams &P, const TileSmem &sm, int e, const Rand4 r)
{
    const float *fr = &sm.frame[e * kFrameStride];
    const int kind = sm.kind[e];
    Photon ph;
    ph.tag = (kind == KIND_CHER_AXIS || kind == KIND_CHER_GEN) ? 0 : 1;
    ph.axis = (kind == KIND_CHER_AXIS);
    // Cherenkov kinds: r holds the photon's two words (cherenkov_words); fluorescence: the four words of its own block
    ph.u3 = (ph.tag == 0) ? cherenkov_u3(r.r0, r.r1) : uniform01(r.r2);
    if (kind == KIND_CHER_AXIS) {
        const float w1 = one_two(r.r0);
        const float sd = fmaf(w1, fr[F_NEGL], fr[F_K0C]);                            // K0 - u1 L
        float sp, cp;
        __sincosf(fmaf(one_two(r.r1), 6.2831853f, -9.42477760f), &sp, &cp);          // phi - pi, in [-pi, pi)
        ph.vz = fmaf(cp, fr[F_AZ], fmaf(sp, fr[F_BZ], fr[F_CZ]));
        ph.vx = fmaf(cp, fr[F_AX], fmaf(sp, fr[F_BX], fr[F_CX]));
        ph.vy = fmaf(cp, fr[F_AY], fmaf(sp, fr[F_BY], fr[F_CY]));
        ph.rva = rcp_approx(ph.vz);
        const float rho = sd * ph.rva;
        ph.gx = fmaf(rho, fmaf(cp, fr[F_PX], sp * fr[F_QX]), fr[F_GX]);
        ph.gy = fmaf(rho, fmaf(cp, fr[F_PY], sp * fr[F_QY]), fr[F_GY]);
        ph.s = (w1 - kOneMinus) * fr[F_LEN];
        ph.ez = -sd * fr[F_DZ];                                                      // emission altitude above z_ref
        ph.ex = ph.ey = 0.0f;
        return ph;
    }
    ph.s = uniform01(r.r0) * fr[F_L];
    ph.ex = fmaf(ph.s, fr[F_D0 + 0], fr[F_E0 + 0]); ph.ey = fmaf(ph.s, fr[F_D0 + 1], fr[F_E0 + 1]);
    ph.ez = fmaf(ph.s, fr[F_D0 + 2], fr[F_E0 + 2]);
    // sin', cos' of phi - pi = pi (2 u2 - 1); 2 u2 - 1 is exact in fp32 (R5)
    float sp, cp;
    sincospi_unit(fmaf(2.0f, uniform01(r.r1), -1.0f), &sp, &cp);
    if (kind == KIND_FL_ISO) {
        // R16: cos(theta) = 1 - 2 u4, v = (cos phi sin th, sin phi sin th, -cos th); cos phi = -cos'
        const float u4 = uniform01(r.r3);
        const float cth = fmaf(-2.0f, u4, 1.0f), uu = u4 * (1.0f - u4), sth = 2.0f * uu * rsqrtf(uu);   // u4 in (0, 1): uu > 0
        ph.vx = -cp * sth; ph.vy = -sp * sth; ph.vz = -cth;
    } else {
        float sth = 1.0f, cth = 1.0f;
        if (kind == KIND_CONE) {                      // R14: 1 - cos(theta') uniform in [0, 1 - cos(alpha_b)]
            const float t = uniform01(r.r3) * fr[F_OMC];
            cth = 1.0f - t; sth = sqrtf(t * (2.0f - t));     // beamed: sin(theta') sets the aim at 10 km, keep the IEEE root
        }
        if constexpr (DISP) {
            if (kind == KIND_CHER_GEN) {
                // n(x) - 1 = eta' = eta (1 + b x^2), x = 1 / lambda; sin^2 = q / (beta n)^2 with
                // q = 2 eta' + eta'^2 - (1 + eta')^2 / gamma^2.  Near the threshold q is a small difference of 2 eta' and
                // 1 / gamma^2, each ~1e-4: in double (head + tail of eta and 1 / gamma^2 from the frame), so that the weight
                // factor keeps the 1e-5 of the parity criterion.
                const float x = fmaf(-ph.u3, P.dinv_lam, P.inv_lam1);
                const double eta = (double)fr[F_DETA] + (double)fr[F_DETA_LO], ig2 = (double)fr[F_DIG2] + (double)fr[F_DIG2_LO];
                const double etap = eta * (1.0 + (double)(P.cauchy_b_f * x) * (double)x), n1 = 1.0 + etap;
                const double q = 2.0 * etap + etap * etap - n1 * n1 * ig2, bn2 = (1.0 - ig2) * n1 * n1;
                const float s2 = (float)(q / bn2);
                sth = sqrtf(fmaxf(s2, 0.0f)); cth = rsqrtf((float)bn2);
                ph.vx = fmaf(sth, fmaf(cp, fr[F_A0 + 0], sp * fr[F_B0 + 0]), cth * fr[F_C0 + 0]);
                ph.vy = fmaf(sth, fmaf(cp, fr[F_A0 + 1], sp * fr[F_B0 + 1]), cth * fr[F_C0 + 1]);
                ph.vz = fmaf(sth, fmaf(cp, fr[F_A0 + 2], sp * fr[F_B0 + 2]), cth * fr[F_C0 + 2]);
                ph.gx = ph.gy = 0.0f;
                ph.rva = (q > 0.0) ? s2 * fr[F_DINVM] : 0.0f;
                return ph;
            }
        }
        ph.vx = fmaf(sth, fmaf(cp, fr[F_A0 + 0], sp * fr[F_B0 + 0]), cth * fr[F_C0 + 0]);
        ph.vy = fmaf(sth, fmaf(cp, fr[F_A0 + 1], sp * fr[F_B0 + 1]), cth * fr[F_C0 + 1]);
        ph.vz = fmaf(sth, fmaf(cp, fr[F_A0 + 2], sp * fr[F_B0 + 2]), cth * fr[F_C0 + 2]);
    }
    ph.gx = ph.gy = ph.rva = 0.0f;
    return ph;
}

__device__ __forceinline__ uint32_t kind_tag(int kind) { return (kind == KIND_CHER_AXIS || kind == KIND_CHER_GEN) ? 0u : 1u; }

// a2 + a3 for photon j of emitter e, any kind (used by the queue drain, the wide test and the generic kinds' hot path).
template <bool DISP = false>
__device__ __forceinline__ Photon make_photon(const KParams &P, const TileSmem &sm, int e, uint32_t j, unsigned long long S)
{
    const uint32_t tag = kind_tag(sm.kind[e]);
    const Rand4 blk = philox4x32_10(P, tag ? j : (j >> 1), (uint32_t)S, (uint32_t)(S >> 32), tag);
    return photon_from_rand<DISP>(P, sm, e, tag ? blk : cherenkov_words(blk, j));
}

// One accepted (photon, telescope) pair, ready for the tally / record.
struct Hit { float x, y, vx, vy, t, lam, w; int k; bool ok; };

// 2^x, MUFU.EX2 alone (flush-to-zero: the arguments here are -h / c log2(e), far from the denormal range)
__device__ __forceinline__ float ex2_approx(float x)
{
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// The pieces of the exact evaluation that evaluate_pair and the dense loop's fast path share.  Every multiply-add is
// an explicit fmaf, so that both callers compile to the same arithmetic and a photon's record does not depend on the
// path that produced it.
//
// Index of the atmosphere layer at altitude habs: from the frame when the segment lies in one layer or two adjacent
// ones (the second from h_next on), else looked up (unused layers carry h_lo = +inf, so the count is the index).
__device__ __forceinline__ int emission_layer(const KParams &P, int li_frame, float h_next, float habs)
{
    int li = li_frame + ((habs >= h_next) ? 1 : 0);
    if (li_frame < 0) {
        li = 0;
#pragma unroll
        for (int i = 1; i < kMaxLayers; ++i) li += (habs >= P.layerf[i].h_lo) ? 1 : 0;
    }
    return li;
}

// Column depth T(h) = a + b exp(-h / c) of layer lf [g/cm^2]; *E = exp(-h / c)
__device__ __forceinline__ float depth_at(const LayerF lf, float habs, float *E)
{
    *E = ex2_approx(-habs * lf.k2);
    return fmaf(lf.b, *E, lf.a);
}

// R8: arrival time = emission time + (geometric path + integral of eta dl) / c,  integral = kappa (T(c_z) - T(e_z)) / |v_z|
__device__ __forceinline__ float arrival_time(const KParams &P, float s, float ibc, float t0, float s_pl, float telT, float Te, float rv)
{
    const float excess = (P.kappa_m * (telT - Te)) * fabsf(rv);
    return fmaf(s_pl + excess, 1.0f / 0.299792458f, fmaf(s, ibc, t0));
}

// R4: Cherenkov wavelength, 1 / lambda uniform
__device__ __forceinline__ float cherenkov_lambda(const KParams &P, float u3) { return rcp_refined(fmaf(-u3, P.dinv_lam, P.inv_lam1)); }

// R10 for an axis-kind photon and coplanar telescopes: q = g - c on the plane z_ref, b^2 = |q|^2 - (q.v)^2, emission
// above the plane, closest approach ahead.
__device__ __forceinline__ bool axis_test_coplanar(float qx, float qy, float vx, float vy, float ez, float rv, float R2, float *s_pl)
{
    const float qv = fmaf(qx, vx, qy * vy);
    const float b2 = fmaf(-qv, qv, fmaf(qx, qx, qy * qy));
    *s_pl = -ez * rv;
    return (b2 <= R2) && (ez > 0.0f) && (*s_pl - qv > 0.0f);
}

// a4 exact test (R10) + arrival time, wavelength, weight for photon `ph` against telescope k.  Only h.ok and h.k are
// defined when the pair is no hit.  COPLANAR (every telescope centre on the plane z_ref: T.z = 0) drops the terms
// that vanish; the values are the same, bit for bit, as those of the general form (x + 0 = x), so a photon's record
// does not depend on which instance evaluated it.
template <int TELSRC, bool COPLANAR = false>
__device__ __forceinline__ Hit evaluate_pair(const KParams &P, const TileSmem &sm, int e, const Photon &ph, int k)
{
    Hit h;
    h.k = k; h.vx = ph.vx; h.vy = ph.vy; h.ok = false;
    if (!(ph.vz < 0.0f)) return h;
    const float4 T = tel_at<TELSRC>(P, k);
    // 1 / v_z to 1 ulp: Newton step on MUFU.RCP (the axis kind brings the MUFU value it projected with)
    const float r0 = ph.axis ? ph.rva : rcp_approx(ph.vz);
    const float rv = fmaf(r0, fmaf(-ph.vz, r0, 1.0f), r0);
    const float *fr = &sm.frame[e * kFrameStride];
    const float habs = P.z_ref_f + ph.ez;
    // Column depth T(e_z) of the emission altitude (R8) and, for R27, the refractivity there.  The layer: the preamble
    // left it in the frame when the whole segment lies in one layer (F_LAYER >= 0), else it is looked up (unused
    // layers carry h_lo = +inf, so the count is the index).
    float Te, eta_e;
    auto atmosphere_at_emission = [&]() {
        const LayerF lf = P.layerf[emission_layer(P, __float_as_int(fr[F_LAYER]), fr[F_HNEXT], habs)];
        float E;
        Te = depth_at(lf, habs, &E);
        eta_e = P.kappa_m * lf.b * (lf.k2 * 0.693147181f) * E;   // eta0 rho(h) / rho0, rho = (b / c) exp(-h / c) / 100
    };
    float s_pl;
    if ((P.flags & kFlagRefract) && ph.vz <= -kRefractVzMin) {
        // R27: point and direction on the plane z = c_z corrected for refraction to first order, then
        // the sphere test on the corrected values.  (x, y) = straight-line plane point relative to the centre.
        float x, y, hk;
        if (ph.axis) {
            hk = ph.ez - T.z;
            x = fmaf(T.z * rv, ph.vx, ph.gx - T.x); y = fmaf(T.z * rv, ph.vy, ph.gy - T.y);
        } else {
            const float mx = T.x - ph.ex, my = T.y - ph.ey, mz = T.z - ph.ez;
            hk = -mz;
            x = fmaf(mz * rv, ph.vx, -mx); y = fmaf(mz * rv, ph.vy, -my);
        }
        if (!(hk > 0.0f)) return h;
        s_pl = -hk * rv;
        atmosphere_at_emission();
        const float arv = fabsf(rv);
        // dr along the horizontal flight direction: (v_x, v_y) / sin(theta0) * tan(theta0) / cos^2(theta0) [...]
        const float G = (eta_e * hk - P.kappa_m * (telT_at<TELSRC>(P, k) - Te)) * arv * arv * arv;
        x = fmaf(ph.vx, G, x); y = fmaf(ph.vy, G, y);
        // dtheta = tan(theta0) f, f = eta(e_z) - eta(c_z):  sin(theta0 + dtheta) = sin(theta0) (1 + f),
        // -cos(theta0 + dtheta) = v_z + sin^2(theta0) f / |v_z|   (second order ~1e-11 dropped)
        const float f = eta_e - telEta_at<TELSRC>(P, k);
        const float vx = fmaf(ph.vx, f, ph.vx), vy = fmaf(ph.vy, f, ph.vy);
        const float qv = fmaf(x, vx, y * vy);
        const float b2 = fmaf(x, x, y * y) - qv * qv;
        if (!(b2 <= T.w) || !(s_pl - qv > 0.0f)) return h;
        h.x = x; h.y = y; h.vx = vx; h.vy = vy;
    } else {
        if (ph.axis) {
            // q = g - c on the plane z_ref:  b^2 = |q|^2 - (q.v)^2,  the point g is at path length -ez / v_z
            const float qx = ph.gx - T.x, qy = ph.gy - T.y;
            if constexpr (COPLANAR) {
                if (!axis_test_coplanar(qx, qy, ph.vx, ph.vy, ph.ez, rv, T.w, &s_pl)) return h;
                h.x = qx; h.y = qy;
            } else {
                const float qz = -T.z;
                const float qv = fmaf(qx, ph.vx, fmaf(qy, ph.vy, qz * ph.vz));
                const float b2 = fmaf(-qv, qv, fmaf(qx, qx, fmaf(qy, qy, qz * qz)));
                const float hk = ph.ez - T.z;                                      // emission height above the telescope plane
                s_pl = -hk * rv;
                const float s_c = (s_pl - T.z * rv) - qv;
                if (!(b2 <= T.w) || !(hk > 0.0f) || !(s_c > 0.0f)) return h;
                h.x = fmaf(T.z * rv, ph.vx, qx); h.y = fmaf(T.z * rv, ph.vy, qy);  // on the plane z = c_z, relative to the centre (R11)
            }
        } else {
            // no plane projection (ill-conditioned for |v_z| -> 0):  b = |m x v|,  m = c - e
            const float mx = T.x - ph.ex, my = T.y - ph.ey, mz = T.z - ph.ez;
            const float cx = fmaf(my, ph.vz, -(mz * ph.vy)), cy = fmaf(mz, ph.vx, -(mx * ph.vz)), cz = fmaf(mx, ph.vy, -(my * ph.vx));
            const float b2 = fmaf(cx, cx, fmaf(cy, cy, cz * cz));
            const float s_c = fmaf(mx, ph.vx, fmaf(my, ph.vy, mz * ph.vz));
            if (!(b2 <= T.w) || !(mz < 0.0f) || !(s_c > 0.0f)) return h;
            s_pl = mz * rv;
            h.x = fmaf(s_pl, ph.vx, -mx); h.y = fmaf(s_pl, ph.vy, -my);
        }
        atmosphere_at_emission();
    }
    h.t = arrival_time(P, ph.s, fr[F_IBC], fr[F_T0], s_pl, telT_at<TELSRC>(P, k), Te, rv);
    // R4: wavelength
    const float u3 = ph.u3;
    h.lam = (ph.tag == 0) ? cherenkov_lambda(P, u3) : fmaf(u3, P.fl_dlam, P.fl_lam1);
    // R17: transmission weight exp(-tau(h, lambda) / |v_z|)
    h.w = fr[F_W0];
    if constexpr (tel_disp(TELSRC)) { if (ph.tag == 0) h.w *= ph.rva; }      // R30: sin^2(lambda) / <sin^2>
    if (P.tau != nullptr) {
        const int nh = P.tau_nh, nl = P.tau_nl;
        float fh = (habs - P.tau_h0) * P.tau_inv_dh, fl = (h.lam - P.tau_l0) * P.tau_inv_dl;
        fh = fminf(fmaxf(fh, 0.0f), (float)(nh - 1)); fl = fminf(fmaxf(fl, 0.0f), (float)(nl - 1));
        const int ih = min(max((int)floorf(fh), 0), max(nh - 2, 0)), il = min(max((int)floorf(fl), 0), max(nl - 2, 0));
        const float th = fh - (float)ih, tl = fl - (float)il;
        const int ih1 = (nh > 1) ? ih + 1 : ih, il1 = (nl > 1) ? il + 1 : il;
        const float t00 = __ldg(&P.tau[ih * nl + il]), t01 = __ldg(&P.tau[ih * nl + il1]);
        const float t10 = __ldg(&P.tau[ih1 * nl + il]), t11 = __ldg(&P.tau[ih1 * nl + il1]);
        const float tau = (1.0f - th) * fmaf(tl, t01 - t00, t00) + th * fmaf(tl, t11 - t10, t10);
        h.w *= __expf(-tau * fabsf(rv));
    }
    h.ok = true;
    return h;
}

// ------------------------------------------------------------------------------------
// Flat photons.  A photon with |v_z| < kFlatVz (isotropic / beamed fluorescence seen from the side, Cherenkov light of a
// horizontal track) travels |c_z - e_z| / |v_z| to the plane of the telescope: kilometres for metres of height.  fp32
// cannot carry it to north_star's 1 cm / 0.1 ns (delta(1 / v_z) = delta v_z / v_z^2), so such a photon only passes a
// conservative fp32 distance test here and is then evaluated in DOUBLE from the segment record: preamble, uniforms from
// the same Philox words, direction, R10, R8, R4, R17.  They are well below 1e-3 of the photons that reach this point.
constexpr float kFlatVz = 0.05f;

__device__ __forceinline__ double column_depth_d(const KParams &P, double h)
{
    const LayerD l = P.layer[layer_of(P, h)];
    return l.a + l.b * exp(-h / l.c);
}

template <bool DISP>
__device__ __noinline__ Hit flat_hit_f64(const KParams &P, unsigned long long S, uint32_t tag, uint32_t j, int k)
{
    Hit h;
    h.ok = false; h.k = k; h.x = h.y = h.vx = h.vy = h.t = h.lam = h.w = 0.0f;
    const float4 *sp = P.seg + (S - P.first_id) * 3ull;
    const float4 s0 = __ldg(sp), s1 = __ldg(sp + 1), s2 = __ldg(sp + 2);
    float scratch[kFrameStride];
    uint8_t kind8;
    int bad;
    bool culled;
    FrameD f;
    [[maybe_unused]] FrameDisp fx;
    const uint32_t nb = preamble<true, false, DISP>(P, s0, s1, s2, (int)tag, scratch, &kind8, &bad, &culled, &f, nullptr, &fx);
    if (bad || culled || j >= nb) return h;
    // a2, R19: U = ((r >> 9) + 1/2) 2^-23; the Cherenkov wavelength uniform from the 9 + 9 low bits (R20)
    const Rand4 blk = philox4x32_10(P, tag ? j : (j >> 1), (uint32_t)S, (uint32_t)(S >> 32), tag);
    const Rand4 r = tag ? blk : cherenkov_words(blk, j);
    const double u1 = ((double)(r.r0 >> 9) + 0.5) * 1.1920928955078125e-07, u2 = ((double)(r.r1 >> 9) + 0.5) * 1.1920928955078125e-07;
    const double u3 = tag ? ((double)(r.r2 >> 9) + 0.5) * 1.1920928955078125e-07
                          : ((double)(((r.r0 & 511u) << 9) | (r.r1 & 511u)) + 0.5) * 3.814697265625e-06;
    const double u4 = ((double)(r.r3 >> 9) + 0.5) * 1.1920928955078125e-07;
    // a3: emission point and time, direction
    const double s = u1 * f.L;
    const double e[3] = { f.p0[0] + s * f.d[0], f.p0[1] + s * f.d[1], f.p0[2] + s * f.d[2] };
    const double t_e = f.t0 + s * f.ibc;
    double sphi, cphi;
    sincos(6.283185307179586476925 * u2, &sphi, &cphi);
    double v[3];
    [[maybe_unused]] double wfac = 1.0;
    if (f.kind == KIND_FL_ISO) {
        const double cth = 1.0 - 2.0 * u4, sth = 2.0 * sqrt(u4 * (1.0 - u4));
        v[0] = cphi * sth; v[1] = sphi * sth; v[2] = -cth;
    } else {
        double sth = f.sin_c, cth = f.cos_c;                     // Cherenkov (generic projection)
        if (f.kind == KIND_CONE) { const double t = u4 * f.omc; cth = 1.0 - t; sth = sqrt(t * (2.0 - t)); }
        if constexpr (DISP) {
            if (f.kind == KIND_CHER_GEN) {                       // R30: the angle and weight factor of this wavelength
                const double x = P.x1_d - u3 * (P.x1_d - P.x2_d), n = 1.0 + fx.d_eta * (1.0 + P.cauchy_b * x * x);
                const double s2 = 1.0 - 1.0 / (fx.d_beta2 * n * n);
                if (!(s2 > 0.0)) return h;
                sth = sqrt(s2); cth = 1.0 / (sqrt(fx.d_beta2) * n);
                wfac = s2 / fx.d_mean;
            }
        }
        double m0[3], m1[3];
        rodrigues_columns(f.axis, m0, m1);
        // M_Rod (cos phi sth, sin phi sth, -cth) with the third column of M_Rod = -axis
        for (int i = 0; i < 3; ++i) v[i] = sth * (cphi * m0[i] + sphi * m1[i]) + cth * f.axis[i];
    }
    // a4, R10: distance from the sphere centre to the forward ray, as a cross product
    // (ground histogram: the one accept-all detector on the observation level about the core)
    const double4 T = (P.hist != nullptr) ? make_double4(P.x_ref, P.y_ref, P.z_ref, 1e15) : P.telD[k];
    const double m[3] = { T.x - e[0], T.y - e[1], T.z - e[2] };
    if (!(v[2] < 0.0) || !(m[2] < 0.0)) return h;
    const double cx = m[1] * v[2] - m[2] * v[1], cy = m[2] * v[0] - m[0] * v[2], cz = m[0] * v[1] - m[1] * v[0];
    const double s_c = m[0] * v[0] + m[1] * v[1] + m[2] * v[2];
    if (!(cx * cx + cy * cy + cz * cz <= T.w * T.w) || !(s_c > 0.0)) return h;
    const double s_pl = m[2] / v[2];
    // R8, R4, R17
    const double excess = 0.01 * (P.eta0 / P.rho0) * (column_depth_d(P, T.z) - column_depth_d(P, e[2])) / fabs(v[2]);
    const double lam = tag ? P.fl_lam1_d + u3 * (P.fl_lam2_d - P.fl_lam1_d)
                           : 1.0 / (1.0 / P.lam1_d - u3 * (1.0 / P.lam1_d - 1.0 / P.lam2_d));
    double w = f.w0;
    if constexpr (DISP) w *= wfac;
    if (P.tau != nullptr) {
        const int nh = P.tau_nh, nl = P.tau_nl;
        double fh = (e[2] - P.tau_h0_d) / P.tau_dh_d, fl = (lam - P.tau_l0_d) / P.tau_dl_d;
        fh = fmin(fmax(fh, 0.0), (double)(nh - 1)); fl = fmin(fmax(fl, 0.0), (double)(nl - 1));
        const int ih = min(max((int)floor(fh), 0), max(nh - 2, 0)), il = min(max((int)floor(fl), 0), max(nl - 2, 0));
        const double th = fh - (double)ih, tl = fl - (double)il;
        const int ih1 = (nh > 1) ? ih + 1 : ih, il1 = (nl > 1) ? il + 1 : il;
        const double t00 = __ldg(&P.tau[ih * nl + il]), t01 = __ldg(&P.tau[ih * nl + il1]);
        const double t10 = __ldg(&P.tau[ih1 * nl + il]), t11 = __ldg(&P.tau[ih1 * nl + il1]);
        const double tau = (1.0 - th) * (t00 + tl * (t01 - t00)) + th * (t10 + tl * (t11 - t10));
        w *= exp(-tau / fabs(v[2]));
    }
    h.x = (float)(e[0] + s_pl * v[0] - T.x); h.y = (float)(e[1] + s_pl * v[1] - T.y);
    h.vx = (float)v[0]; h.vy = (float)v[1];
    h.t = (float)(t_e + (s_pl + excess) * (1.0 / 0.299792458));
    h.lam = (float)lam; h.w = (float)w;
    h.ok = true;
    return h;
}

// evaluate_pair, with the flat photons of the generic kinds set aside for flat_hit_f64 once they pass a conservative
// fp32 distance test (cross product, no plane projection, slack for the fp32 error): the pair goes to the tile's flat list,
// which is worked off in double after the photon loops (flat_pass) -- the loops themselves never call into the
// double-precision code, whose register needs would otherwise spill their state.  j = photon index.  A full list
// (more than kFlatList such pairs in one tile: not seen in any config) leaves the pair to fp32.  The ground histogram
// keeps fp32 throughout: a flat photon lands beyond 20 times its emission height, far outside any profile.
template <int TELSRC, bool COPLANAR = false>
__device__ __forceinline__ Hit evaluate_any(const KParams &P, TileSmem &sm, int e, const Photon &ph, int k, uint32_t j)
{
    if (!ph.axis && ph.vz > -kFlatVz && P.hist == nullptr) {
        Hit h;
        h.ok = false; h.k = k;
        if (!(ph.vz < 0.0f)) return h;
        const float4 T = tel_at<TELSRC>(P, k);
        if (!(T.w > 0.0f)) return h;                                   // an unused constant-bank slot (R^2 = -1)
        const float mx = T.x - ph.ex, my = T.y - ph.ey, mz = T.z - ph.ez;
        const float cx = fmaf(my, ph.vz, -(mz * ph.vy)), cy = fmaf(mz, ph.vx, -(mx * ph.vz)), cz = fmaf(mx, ph.vy, -(my * ph.vx));
        const float b2 = fmaf(cx, cx, fmaf(cy, cy, cz * cz)), mm = fmaf(mx, mx, fmaf(my, my, mz * mz));
        // fp32 error of b = |m x v|: |m| delta v (~3e-7) + delta m (1 ulp of a coordinate ~ 1e-7 |m|): below 1e-6 |m|
        const float thr = sqrtf(T.w) + fmaf(2e-6f, sqrtf(mm), 2e-3f);
        if (!(b2 <= thr * thr)) return h;
        const uint32_t slot = atomicAdd(&sm.flat_count, 1u);
        if (slot < (uint32_t)kFlatList) { sm.flat_list[slot] = make_uint2(j | ((uint32_t)e << 24), (uint32_t)k); return h; }
    }
    return evaluate_pair<TELSRC, COPLANAR>(P, sm, e, ph, k);
}

__device__ __forceinline__ unsigned long long emitter_segment(const KParams &P, unsigned long long tile_first, int e)
{
    return tile_first + (unsigned)((P.n_procs == 2) ? (e & (kTile / 2 - 1)) : e);
}

// The tile's flat list in double (see evaluate_any), by all threads of the tile after the photon loops: tally, record.
template <int MODE, bool DISP>
__device__ __noinline__ void flat_pass(const KParams &P, TileSmem &sm, unsigned long long tile_first)
{
    const uint32_t n = min(sm.flat_count, (uint32_t)kFlatList);
    for (uint32_t i = threadIdx.x; i < n; i += kTile) {
        const uint2 q = sm.flat_list[i];
        const int e = (int)(q.x >> 24), k = (int)q.y;
        const uint32_t j = q.x & 0xffffffu, tag = kind_tag(sm.kind[e]);
        const unsigned long long S = emitter_segment(P, tile_first, e);
        const Hit h = flat_hit_f64<DISP>(P, S, tag, j, k);
        if (!h.ok) continue;
        const double w = (double)h.w;
        if (P.n_tel <= kTelSmemMax) { atomicAdd(&sm.t_hits[k], 1u); atomicAdd(&sm.t_sw[k], w); atomicAdd(&sm.t_swt[k], w * (double)h.t); }
        else { atomicAdd(&P.tallies[k].hits, 1ull); atomicAdd(&P.tallies[k].sum_w, w); atomicAdd(&P.tallies[k].sum_wt, w * (double)h.t); }
        if constexpr (MODE == MODE_OUT) {
            const unsigned long long slot = atomicAdd(&P.cursors[k], 1ull);
            if (slot < P.tel_capacity[k]) {
                const unsigned long long at = P.tel_offset[k] + slot;
                float *rec = P.records + at * (unsigned)kRecWords;
                rec[0] = h.x; rec[1] = h.y; rec[2] = h.vx; rec[3] = h.vy; rec[4] = h.t; rec[5] = h.lam; rec[6] = h.w;
                if (P.ids) P.ids[at] = (S << 25) | ((unsigned long long)tag << 24) | (unsigned long long)j;
            }
        }
    }
}

// Photon output, hits on several telescopes: the lanes of one telescope reserve their records with a single bump of
// that telescope's cursor.  Called by all 32 lanes.
__device__ __forceinline__ void write_records_grouped(const KParams &P, const Hit &h, uint64_t id)
{
    const uint32_t lane = lane_id();
    const uint32_t peers = __match_any_sync(0xffffffffu, h.ok ? h.k : -1 - (int)lane);
    if (h.ok) {
        const int leader = __ffs(peers) - 1;
        unsigned long long base = 0;
        if ((int)lane == leader) base = atomicAdd(&P.cursors[h.k], (unsigned long long)__popc(peers));
        base = __shfl_sync(peers, base, leader);
        const unsigned long long slot = base + (unsigned)__popc(peers & ((1u << lane) - 1u));
        if (slot < P.tel_capacity[h.k]) {
            const unsigned long long at = P.tel_offset[h.k] + slot;
            float *rec = P.records + at * (unsigned)kRecWords;
            rec[0] = h.x; rec[1] = h.y; rec[2] = h.vx; rec[3] = h.vy; rec[4] = h.t; rec[5] = h.lam; rec[6] = h.w;
            if (P.ids) P.ids[at] = id;
        }
    }
}

// Tally: a thread adds its hits to its own accumulator in shared memory (no shuffles, no atomics)
// and flushes it into the tile tallies when the telescope changes and at the end of the tile.
__device__ __forceinline__ void flush_accumulator(const KParams &P, TileSmem &sm)
{
    const int t = threadIdx.x;
    const uint32_t n = sm.acc_n[t];
    if (n == 0u) return;
    const int k = sm.acc_k[t];
    if (P.n_tel <= kTelSmemMax) { atomicAdd(&sm.t_hits[k], n); atomicAdd(&sm.t_sw[k], sm.acc_w[t]); atomicAdd(&sm.t_swt[k], sm.acc_wt[t]); }
    else { atomicAdd(&P.tallies[k].hits, (unsigned long long)n); atomicAdd(&P.tallies[k].sum_w, sm.acc_w[t]); atomicAdd(&P.tallies[k].sum_wt, sm.acc_wt[t]); }
    sm.acc_n[t] = 0u; sm.acc_w[t] = 0.0; sm.acc_wt[t] = 0.0;
}

__device__ __forceinline__ void accumulate_hit(const KParams &P, TileSmem &sm, const Hit &h)
{
    const int t = threadIdx.x;
    if (sm.acc_k[t] != h.k) { flush_accumulator(P, sm); sm.acc_k[t] = h.k; }
    const double w = (double)h.w;
    sm.acc_n[t] += 1u; sm.acc_w[t] += w; sm.acc_wt[t] += w * (double)h.t;
}

// Photon output when all hits of the warp are on one telescope k0 (okm = the lanes holding one): one bump of that
// telescope's cursor for the warp (sparse tiles, queue drains, telescopes other than a dense tile's own).
__device__ __forceinline__ void write_records_one_tel(const KParams &P, const Hit &h, uint64_t id, uint32_t okm, int k0)
{
    const uint32_t lane = lane_id();
    const uint32_t n = (uint32_t)__popc(okm), rank = (uint32_t)__popc(okm & ((1u << lane) - 1u));
    unsigned long long base = 0;
    if (lane == 0u) base = atomicAdd(&P.cursors[k0], (unsigned long long)n);
    base = __shfl_sync(0xffffffffu, base, 0);
    const unsigned long long cap = P.tel_capacity[k0];
    if (base >= cap) return;
    if (h.ok && base + rank < cap) {
        const unsigned long long at = P.tel_offset[k0] + base + rank;
        float *rec = P.records + at * (unsigned)kRecWords;
        rec[0] = h.x; rec[1] = h.y; rec[2] = h.vx; rec[3] = h.vy; rec[4] = h.t; rec[5] = h.lam; rec[6] = h.w;
        if (P.ids) P.ids[at] = id;
    }
}

// mbarrier and acq_rel add on shared memory, CTA scope (the reservation rounds of the dense loop)
__device__ __forceinline__ void mbar_init(unsigned long long *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_release(unsigned long long *bar)
{
    asm volatile("mbarrier.arrive.release.cta.shared::cta.b64 _, [%0];" :: "r"((uint32_t)__cvta_generic_to_shared(bar)) : "memory");
}
// wait until the phase of the given parity has completed (acquire); the hardware suspends the thread between tries
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.acquire.cta.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "nanosleep.u32 200;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" :: "r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ uint32_t add_acq_rel_cta(uint32_t *p, uint32_t v)
{
    uint32_t old;
    asm volatile("atom.acq_rel.cta.shared.add.u32 %0, [%1], %2;" : "=r"(old) : "r"((uint32_t)__cvta_generic_to_shared(p)), "r"(v) : "memory");
    return old;
}

// Dense tiles: copy the block of n records a warp staged in round r (words [0, 7 n) at st) to the slots the round
// reserved for it, [base_r + off, base_r + off + n) of the dense telescope's region (cap records from global record
// slot tel_off on).  Waits (every lane polls the flag in shared memory: a broadcast read, no divergence) until the
// last arrival of round r has published base_r; a whole round of arithmetic lies between the warp's own arrival and
// this call, so the wait is normally over.  Called by all 32 lanes, every round, also with n == 0: the wait is what
// keeps a warp from running more than kRoundSlots - 1 rounds ahead of the others.
//
// 16-byte stores: record slot s starts at word 7 s, so the words of a shared-memory slot and of a global slot are in
// the same position within a 16-byte vector iff the two slot numbers agree modulo 4.  The order of the records
// within a region is free (R22), so the block is rotated by rho = (-G) mod 4 slots, G = first global slot: staged
// slot s goes to global slot G + rho + s, whose address is a multiple of 16 bytes for s = 0 -- the body is copied as
// aligned float4 vectors, 512 contiguous bytes per store instruction -- and the last rho (<= 3) staged records wrap
// around to global slots G .. G + rho - 1 as scalar words, together with the <= 3 words the body leaves over.
template <int SUB, bool IDS>
__device__ __forceinline__ void copy_block(const KParams &P, OutSmem &os, const float *st, const unsigned long long cap,
                                           const unsigned long long tel_off, const uint32_t n, const uint32_t off, const uint32_t r)
{
    const uint32_t lane = lane_id();
    mbar_wait(&os.rbar[r & (kRoundSlots - 1)], (r / (uint32_t)kRoundSlots) & 1u);
    const unsigned long long first = *(volatile unsigned long long *)&os.rbase[r & (kRoundSlots - 1)] + off;
    if (n == 0u || first >= cap) return;
    const uint32_t m = (uint32_t)min((unsigned long long)n, cap - first);
    const unsigned long long G = tel_off + first;
    float *dst = P.records + G * (unsigned)kRecWords;
    const unsigned long long *sid = reinterpret_cast<const unsigned long long *>(st + kBlockRecs * kRecWords);   // general path
    if ((reinterpret_cast<uintptr_t>(P.records) & 15u) == 0u) {
        const uint32_t rho = min((0u - (uint32_t)G) & 3u, m), body = (m - rho) * kRecWords, nvec = body >> 2, rest = body & 3u;
        const float4 *src4 = reinterpret_cast<const float4 *>(st);
        float4 *dst4 = reinterpret_cast<float4 *>(dst + rho * kRecWords);
#pragma unroll
        for (uint32_t v0 = 0; v0 < (uint32_t)(SUB * kBlockRecs * kRecWords) / 4u; v0 += 32u) {
            const uint32_t v = v0 + lane;
            if (v < nvec) __stcs(&dst4[v], src4[v]);
        }
        // lanes 0 .. 7 rho - 1: the wrapped records; the next `rest` lanes: the words the vectors left over
        const uint32_t nwrap = rho * kRecWords;
        if (lane < nwrap) dst[lane] = st[body + lane];
        else if (lane < nwrap + rest) dst[lane + (body - rest)] = st[lane - nwrap + (body - rest)];
        if constexpr (IDS)
            for (uint32_t s = lane; s < m; s += 32u) P.ids[(s < m - rho) ? G + rho + s : G + s - (m - rho)] = sid[s];
    } else {
        const uint32_t nwords = m * kRecWords;
#pragma unroll 4
        for (uint32_t i = lane; i < nwords; i += 32u) dst[i] = st[i];
        if constexpr (IDS)
            for (uint32_t s = lane; s < m; s += 32u) P.ids[G + s] = sid[s];
    }
}

// a5 for up to 32 evaluated pairs, one per lane (h.ok says which lanes hold a hit).  Called by all 32 lanes together.
template <int MODE>
__device__ __forceinline__ void commit_hits(const KParams &P, TileSmem &sm, const Hit &h, uint64_t id)
{
    const uint32_t okm = __ballot_sync(0xffffffffu, h.ok);
    if (okm == 0u) return;
    if constexpr (MODE == MODE_HIST) {
        // ground-plane radial profile: h.x, h.y are relative to the core on the plane z = h_obs
        HistSmem &hs = hist_smem(sm);
        bool over = false;
        if (h.ok) {
            const float r2 = fmaf(h.x, h.x, h.y * h.y);
            const float r = r2 * rsqrtf(fmaxf(r2, 1e-30f));
            const float fb = r * P.hist_inv_dr;
            over = !(fb < (float)P.hist_bins);
            if (!over) {
                const int b = (int)fb;
                const uint32_t qw = min(__float2uint_rn(h.w * P.hist_wscale), 1u << 20);
                const int qt = __float2int_rn(fminf(fmaxf(h.t, -3.0e7f), 3.0e7f) * 64.0f);
                const long long x = (long long)qw * (long long)qt;
                const uint32_t x_lo = (uint32_t)x, x_hi = (uint32_t)((unsigned long long)x >> 32);
                atomicAdd(&hs.n[b], 1u);
                if (atomicAdd(&hs.sw_lo[b], qw) + qw < qw) atomicAdd(&hs.sw_hi[b], 1u);
                const uint32_t carry = (atomicAdd(&hs.swt_lo[b], x_lo) + x_lo < x_lo) ? 1u : 0u;
                if (x_hi + carry) atomicAdd(&hs.swt_hi[b], x_hi + carry);
            }
        }
        const uint32_t om = __ballot_sync(0xffffffffu, over);
        if (om && lane_id() == 0u) atomicAdd(&hs.overflow, (uint32_t)__popc(om));
        return;
    }
    if (h.ok) accumulate_hit(P, sm, h);
    if constexpr (MODE == MODE_OUT) {
        const int k0 = __shfl_sync(0xffffffffu, h.k, __ffs(okm) - 1);
        if (__all_sync(0xffffffffu, !h.ok || h.k == k0)) write_records_one_tel(P, h, id, okm, k0);
        else write_records_grouped(P, h, id);
    }
}

// ---- the per-warp candidate queue.  Entry = (emitter, photon index, telescope) in 8 bytes:
// x = j (24 bits) | e << 24,  y = telescope index.  The warp-uniform count lives in a register.

template <int TELSRC, int MODE>
__device__ __noinline__ void drain_queue(const KParams &P, TileSmem &sm, unsigned long long tile_first, uint32_t head, uint32_t n)
{
    // lanes 0 .. n-1 take one entry each; the others only take part in the warp-wide commit
    const uint32_t lane = lane_id(), warp = threadIdx.x >> 5;
    Hit h;
    h.ok = false; h.k = 0; h.x = h.y = h.vx = h.vy = h.t = h.lam = h.w = 0.0f;
    uint64_t id = 0;
    if (lane < n) {
        const uint2 q = sm.queue[warp][(head + lane) & (kQueue - 1)];
        const int e = (int)(q.x >> 24);
        const uint32_t j = q.x & 0xffffffu;
        const unsigned long long S = emitter_segment(P, tile_first, e);
        const Photon ph = make_photon<tel_disp(TELSRC)>(P, sm, e, j, S);
        h = evaluate_any<TELSRC>(P, sm, e, ph, (int)q.y, j);
        id = (S << 25) | ((unsigned long long)ph.tag << 24) | (unsigned long long)j;
    }
    __syncwarp();
    commit_hits<MODE>(P, sm, h, id);
}

// Dense path: when at least kDenseMin lanes of a warp iteration hold a candidate, the pairs are evaluated on the spot
// from the random words the lanes still hold (no queue, no second Philox).  `has` says which lanes take part; all 32 call.
template <int TELSRC, int MODE>
__device__ __noinline__ void dense_eval(const KParams &P, TileSmem &sm, unsigned long long tile_first, int e, uint32_t j,
                                        uint32_t r0, uint32_t r1, uint32_t r2, uint32_t r3, int k, bool has)
{
    Hit h;
    h.ok = false; h.k = 0; h.x = h.y = h.vx = h.vy = h.t = h.lam = h.w = 0.0f;
    uint64_t id = 0;
    if (has) {
        const unsigned long long S = emitter_segment(P, tile_first, e);
        const Photon ph = photon_from_rand<tel_disp(TELSRC)>(P, sm, e, Rand4{r0, r1, r2, r3});
        h = evaluate_any<TELSRC>(P, sm, e, ph, k, j);
        id = (S << 25) | ((unsigned long long)ph.tag << 24) | (unsigned long long)j;
    }
    __syncwarp();
    commit_hits<MODE>(P, sm, h, id);
}

// Push the candidates of this iteration (per lane: bit c of `cm` set = candidate number c, whose telescope
// index is tel_of(c)) and drain 32 entries whenever that many are queued.  All 32 lanes call it together.
template <int TELSRC, int MODE, typename TelOf>
__device__ __forceinline__ void push_candidates(const KParams &P, TileSmem &sm, unsigned long long tile_first,
                                                uint32_t &q_head, uint32_t &q_count, uint32_t cm, int e, uint32_t j, TelOf tel_of)
{
    const uint32_t lane = lane_id(), warp = threadIdx.x >> 5;
    while (true) {
        const uint32_t have = __ballot_sync(0xffffffffu, cm != 0u);
        if (have == 0u) break;
        if (cm != 0u) {
            const int c = __ffs(cm) - 1;
            cm &= cm - 1u;
            const uint32_t pos = q_head + q_count + (uint32_t)__popc(have & ((1u << lane) - 1u));
            sm.queue[warp][pos & (kQueue - 1)] = make_uint2(j | ((uint32_t)e << 24), (uint32_t)tel_of(c));
        }
        q_count += (uint32_t)__popc(have);
        __syncwarp();
        if (q_count >= 32u) {
            drain_queue<TELSRC, MODE>(P, sm, tile_first, q_head, 32u);
            __syncwarp();
            q_head = (q_head + 32u) & (kQueue - 1);
            q_count -= 32u;
        }
    }
}

// ---- conservative pre-tests on the crossing (gx, gy) of the plane z_ref (valid while |v_z| is not tiny).
// Coplanar telescopes (q_z = 0): b^2 >= |q|^2 v_z^2, so |q|^2 v_z^2 (1 - 1e-4) > R^2 is a miss.
// `add` widens the test for the refraction corrections (R27): a point that moves by at most d in the plane can be hit
// if |q| |v_z| <= R + x, x = d |v_z|, and (R + x)^2 <= R^2 + x (2 R_max + x) = R^2 + add.  0 without the flag.
template <bool COPLANAR>
__device__ __forceinline__ bool plane_pretest(const float4 T, float gx, float gy, float vx, float vy, float vz, float vz2s, float add)
{
    const float qx = gx - T.x, qy = gy - T.y;
    if (COPLANAR) return fmaf(fmaf(qy, qy, qx * qx), vz2s, -add) <= T.w;
    const float qv = fmaf(qx, vx, fmaf(qy, vy, -T.z * vz));
    const float qq = fmaf(qx, qx, fmaf(qy, qy, T.z * T.z));
    return qq - qv * qv - add <= fmaf(qq, 1e-5f, fmaf(T.w, 1.0001f, 1e-3f));   // slack for the fp32 cancellation
}

// Slack of the pre-tests for a photon whose arrival point the refraction corrections may move (|v_z| >= kRefractVzMin).
__device__ __forceinline__ float refraction_slack(const KParams &P, float vz)
{
    if (!(vz <= -kRefractVzMin)) return 0.0f;
    const float rv = rcp_approx(vz), s2 = fmaf(-vz, vz, 1.0f);
    const float x = 1.01f * P.refr_cmax * sqrtf(fmaxf(s2, 0.0f)) * rv * rv;      // d |v_z| = cmax sin / cos^2
    return x * (P.refr_two_rmax + x);
}

// How far the refraction corrections can move the arrival point of a photon in the plane (wide test): 0 for |v_z| < kRefractVzMin
__device__ __forceinline__ float refraction_reach(const KParams &P, float vz)
{
    if (!(vz <= -kRefractVzMin)) return 0.0f;
    const float rv = rcp_approx(vz), s2 = fmaf(-vz, vz, 1.0f);
    return 1.02f * P.refr_cmax * sqrtf(fmaxf(s2, 0.0f)) * fabsf(rv * rv * rv) + 0.01f;
}

// Candidate mask of a photon over the telescopes reachable from its plane crossing.
//  TEL_CONST: bit k = telescope k.   TEL_GRID: bit c = slot c of the photon's grid cell (returned in *cell).
//  Photons flatter than the grid allows, and TEL_GLOBAL, return kAllTelescopes: the caller tests all of them.
constexpr uint32_t kAllTelescopes = 0x80000000u;

// telescope index of candidate bit c
template <int TELSRC> __device__ __forceinline__ uint32_t slot_telescope(const uint2 cell, int c)
{
    if (tel_base(TELSRC) == TEL_GRID) return ((c < 2 ? cell.x : cell.y) >> (16 * (c & 1))) & 0xffffu;
    return (uint32_t)c;
}

// Candidates of one grid level: cell of the plane crossing (most cells are empty: one load, one compare), then the
// pre-test of the telescopes listed there (slots fill from 0, so the first empty slot ends the list).
template <bool COPLANAR>
__device__ __forceinline__ uint32_t grid_lookup(const KParams &P, const GridLevel &G, float gx, float gy, float vx, float vy, float vz, uint2 *cell,
                                                float add)
{
    const int ix = __float2int_rd(fmaf(gx, G.inv_cell, G.ox)), iy = __float2int_rd(fmaf(gy, G.inv_cell, G.oy));
    if ((unsigned)ix >= (unsigned)G.nx || (unsigned)iy >= (unsigned)G.ny) return 0u;
    const uint2 c = __ldg(&P.grid[G.base + iy * G.nx + ix]);
    if (c.x == 0xffffffffu) return 0u;
    *cell = c;
    const float vz2s = vz * vz * 0.9999f;
    uint32_t cm = plane_pretest<COPLANAR>(__ldg(&P.telA[c.x & 0xffffu]), gx, gy, vx, vy, vz, vz2s, add) ? 1u : 0u;
    if ((c.x >> 16) != 0xffffu) {
        if (plane_pretest<COPLANAR>(__ldg(&P.telA[c.x >> 16]), gx, gy, vx, vy, vz, vz2s, add)) cm |= 2u;
        if (c.y != 0xffffffffu) {
            if (plane_pretest<COPLANAR>(__ldg(&P.telA[c.y & 0xffffu]), gx, gy, vx, vy, vz, vz2s, add)) cm |= 4u;
            if ((c.y >> 16) != 0xffffu && plane_pretest<COPLANAR>(__ldg(&P.telA[c.y >> 16]), gx, gy, vx, vy, vz, vz2s, add)) cm |= 8u;
        }
    }
    return cm;
}

template <int TELSRC, bool COPLANAR, int NT, bool REFR>
__device__ __forceinline__ uint32_t plane_candidates(const KParams &P, float gx, float gy, float vx, float vy, float vz, uint2 *cell)
{
    if constexpr (tel_base(TELSRC) == TEL_CONST) {
        const float vz2s = vz * vz * 0.9999f, add = REFR ? refraction_slack(P, vz) : 0.0f;
        uint32_t cm = 0u;
        // NT = n_tel rounded up to 1, 4 or 8; the unused slots hold R^2 = -1 (never a candidate).  Unrolled so that the
        // telescope coordinates are constant-bank operands.
#pragma unroll
        for (int k = 0; k < NT; ++k)
            if (plane_pretest<COPLANAR>(P.tel_c[k], gx, gy, vx, vy, vz, vz2s, add)) cm |= 1u << k;
        return cm;
    } else if constexpr (tel_base(TELSRC) == TEL_GRID) {
        // steep photons use level 0; flatter ones the coarser level 1 when it exists, else the wide test.  One code
        // path per level, so that the level's parameters are constant-bank operands.
        if (-vz >= P.grid_lvl[0].vzmin) {
            // with the refraction corrections the steep photons use the copy of level 0 whose discs carry their reach
            if (REFR) return grid_lookup<COPLANAR>(P, P.grid_lvl[kGridLevels], gx, gy, vx, vy, vz, cell, refraction_slack(P, vz));
            return grid_lookup<COPLANAR>(P, P.grid_lvl[0], gx, gy, vx, vy, vz, cell, 0.0f);
        }
        // corrected photons flatter than level 0 serves: their reach (up to 62 refr_cmax) is beyond what a grid of
        // <= 4 telescopes per cell can hold, so they take the wide test, which carries the slack
        if (REFR && -vz >= kRefractVzMin) return kAllTelescopes;
        if (P.n_grid_levels > 1 && -vz >= P.grid_lvl[1].vzmin) return grid_lookup<COPLANAR>(P, P.grid_lvl[1], gx, gy, vx, vy, vz, cell, 0.0f);
        return kAllTelescopes;
    } else {
        return kAllTelescopes;
    }
}

// Wide test (photons flatter than the grids allow under TEL_GRID, every photon under TEL_GLOBAL).  Such photons are
// collected in a per-warp list; a batch of up to 32 is processed with one photon per lane: the lane rebuilds its
// photon from the counter and tests every telescope (the table is read at warp-uniform addresses) with a
// conservative distance test (cross product, no plane projection: valid for any v_z); the survivors go through the
// candidate queue like all others.
template <int TELSRC, int MODE>
__device__ __noinline__ void wide_batch(const KParams &P, TileSmem &sm, unsigned long long tile_first, uint32_t &q_head,
                                        uint32_t &q_count, uint32_t n)
{
    const uint32_t lane = lane_id(), warp = threadIdx.x >> 5;
    int e = 0;
    uint32_t j = 0u;
    bool live = false;
    float px = 0.f, py = 0.f, pz = 0.f, vx = 0.f, vy = 0.f, vz = 0.f;
    if (lane < n) {
        const uint32_t q = sm.wide_list[warp][lane];
        e = (int)(q >> 24); j = q & 0xffffffu;
        const Photon ph = make_photon<tel_disp(TELSRC)>(P, sm, e, j, emitter_segment(P, tile_first, e));
        live = ph.vz < 0.0f;
        // a point of the ray relative to (x_ref, y_ref, z_ref): the plane crossing (axis kind) or the emission point
        px = ph.axis ? ph.gx : ph.ex; py = ph.axis ? ph.gy : ph.ey; pz = ph.axis ? 0.0f : ph.ez;
        vx = ph.vx; vy = ph.vy; vz = ph.vz;
    }
    // R27: the corrections move the ray by at most refr_cmax sin / cos^3 in the plane, so b changes by no more than that
    const float slack = (P.flags & kFlagRefract) ? refraction_reach(P, vz) : 0.0f;
    const float add = slack * (P.refr_two_rmax + slack);
    for (int k0 = 0; k0 < P.n_tel; k0 += 32) {
        uint32_t cm = 0u;
        const int kn = min(32, P.n_tel - k0);
        if (live) {
            for (int c = 0; c < kn; ++c) {
                const float4 T = __ldg(&P.telA[k0 + c]);
                const float mx = T.x - px, my = T.y - py, mz = T.z - pz;
                const float cx = fmaf(my, vz, -(mz * vy)), cy = fmaf(mz, vx, -(mx * vz)), cz = fmaf(mx, vy, -(my * vx));
                const float b2 = fmaf(cx, cx, fmaf(cy, cy, cz * cz));
                const float mm = fmaf(mx, mx, fmaf(my, my, mz * mz));
                if (b2 <= fmaf(mm, 1e-5f, fmaf(T.w, 1.0001f, 1e-3f)) + add) cm |= 1u << c;
            }
        }
        if (__any_sync(0xffffffffu, cm != 0u))
            push_candidates<TELSRC, MODE>(P, sm, tile_first, q_head, q_count, cm, e, j, [&](int c) { return (uint32_t)(k0 + c); });
    }
}

// Append the photons of the lanes in `wide` to the warp's list and process a batch when 32 are waiting.
template <int TELSRC, int MODE>
__device__ __forceinline__ void wide_push(const KParams &P, TileSmem &sm, unsigned long long tile_first, uint32_t &q_head,
                                          uint32_t &q_count, uint32_t wide, int e, uint32_t j)
{
    const uint32_t lane = lane_id(), warp = threadIdx.x >> 5;
    __syncwarp();
    uint32_t n = sm.wide_count[warp];
    if ((wide >> lane) & 1u) sm.wide_list[warp][n + (uint32_t)__popc(wide & ((1u << lane) - 1u))] = j | ((uint32_t)e << 24);
    n += (uint32_t)__popc(wide);
    __syncwarp();
    if (n >= 32u) {
        wide_batch<TELSRC, MODE>(P, sm, tile_first, q_head, q_count, 32u);
        __syncwarp();
        const uint32_t moved = (lane < n - 32u) ? sm.wide_list[warp][32u + lane] : 0u;
        __syncwarp();
        if (lane < n - 32u) sm.wide_list[warp][lane] = moved;
        n -= 32u;
    }
    if (lane == 0u) sm.wide_count[warp] = n;
}

// The polar window of a fluorescence emitter (see the preamble): true = the photon with polar word r3 cannot reach the
// array, or goes up (*up; counted by the caller) -- decided from one uniform, before the direction is built.
__device__ __forceinline__ bool polar_cull(const TileSmem &sm, int e, int kind, uint32_t r3, bool *up)
{
    const float *fr = &sm.frame[e * kFrameStride];
    *up = false;
    if (kind == KIND_FL_ISO) {
        const float vz = fmaf(2.0f, uniform01(r3), -1.0f);             // - cos(theta), exact (R16)
        *up = !(vz < 0.0f);
        return *up || vz < fr[F_VZLO] || vz > fr[F_VZHI];
    }
    if (kind == KIND_CONE) return uniform01(r3) * fr[F_OMC] > fr[F_TMAX];
    return false;
}

// a2-a4 of the hot loop for the generic kinds.  Returns the candidate mask (see plane_candidates); *upward is
// set when the photon does not go down.  Photons flatter than |v_z| = 0.05 are tested against all telescopes.
template <int TELSRC, bool COPLANAR, int NT, bool REFR>
__device__ __noinline__ uint32_t generic_candidates(const KParams &P, const TileSmem &sm, int e, uint32_t r0, uint32_t r1, uint32_t r2,
                                                    uint32_t r3, uint2 *cell, bool *upward)
{
    const Photon ph = photon_from_rand<tel_disp(TELSRC)>(P, sm, e, Rand4{r0, r1, r2, r3});
    if constexpr (tel_disp(TELSRC)) {
        if (ph.tag == 0 && ph.rva == 0.0f) { *upward = false; return 0u; }      // R30: below the threshold at its wavelength
    }
    *upward = !(ph.vz < 0.0f);
    if (*upward) return 0u;
    if (ph.vz > -0.05f) return kAllTelescopes;
    const float spl = -ph.ez * rcp_approx(ph.vz);          // candidate search only: the pre-tests carry slack
    return plane_candidates<TELSRC, COPLANAR, NT, REFR>(P, fmaf(spl, ph.vx, ph.ex), fmaf(spl, ph.vy, ph.ey), ph.vx, ph.vy, ph.vz, cell);
}

// ------------------------------------------------------------------------------------
struct AxisFrame { float negL, k0c, az, bz, cz, px, py, qx, qy, gx, gy; };

__device__ __forceinline__ AxisFrame load_axis_frame(const TileSmem &sm, int e)
{
    const float4 *fp = reinterpret_cast<const float4 *>(&sm.frame[e * kFrameStride]);
    const float4 A = fp[0], B = fp[1], C = fp[2];
    return AxisFrame{A.x, A.y, A.z, A.w, B.x, B.y, B.z, B.w, C.x, C.y, C.z};
}

// ------------------------------------------------------------------------------------
// The lane's position in its warp's photon range and everything else the photon loop carries.
struct WarpWalk {
    int e, kind;                       // current emitter and its kind
    uint32_t end, g, j;                // real end of the emitter in the tile's index space, photon index, index within the emitter
    PhiloxEmitter pe;
    AxisFrame f_reg;
    uint32_t n_up, q_head, q_count;
};

// The photon loop of the grid / global-table photon-output kernels (phase 2): one photon per lane and iteration, its
// half of the Philox block selected by the photon index; candidates go to the queue, or are evaluated on the spot when
// at least kDenseMin lanes hold one.
template <int TELSRC, bool COPLANAR, int NT, int MODE, bool REFR>
__device__ __forceinline__ void walk(const KParams &P, TileSmem &sm, WarpWalk &ww, const uint32_t hi, const unsigned long long tile_first,
                                     const uint32_t n_iter)
{
    constexpr bool kFrameInRegs = (tel_base(TELSRC) == TEL_CONST);
    int e = ww.e, kind = ww.kind;
    uint32_t end = ww.end, g = ww.g, j = ww.j, n_up = ww.n_up, q_head = ww.q_head, q_count = ww.q_count;
    PhiloxEmitter pe = ww.pe;
    AxisFrame f_reg = ww.f_reg;
    for (uint32_t it = 0; it < n_iter; ++it, g += 32u, j += 32u) {
        bool active = g < hi;                        // the lanes past the warp's range idle in its last iterations
        uint32_t cm = 0u;
        uint2 cell = make_uint2(0xffffffffu, 0xffffffffu);
        Rand4 r = {0u, 0u, 0u, 0u};
        if (active) {
            // `end` holds the emitter's real end (its padded end less the empty slot after an odd count)
            if (g >= ((end + 1u) & ~1u)) {
                uint32_t pend;
                do { ++e; pend = sm.prefix[e + 1]; } while (g >= pend);
                end = pend - sm.odd[e];
                j = g - sm.prefix[e];
                kind = sm.kind[e];
                pe = philox_emitter(P, emitter_segment(P, tile_first, e));
                if (kFrameInRegs) f_reg = load_axis_frame(sm, e);
            }
            if (g >= end) active = false;             // the empty slot
        }
        if (active) {
            if (kind == KIND_CHER_AXIS) {
                const AxisFrame f = kFrameInRegs ? f_reg : load_axis_frame(sm, e);
                r = cherenkov_words(philox_photon(P, pe, j >> 1, 0u), j);                      // a2 (R20)
                // a3: remaining axis path length to the plane, azimuth (PAPER.md:61 c_rng, R5)
                const float sd = fmaf(one_two(r.r0), f.negL, f.k0c);                          // K0 - u1 L
                float sp, cp;
                __sincosf(fmaf(one_two(r.r1), 6.2831853f, -9.42477760f), &sp, &cp);           // phi - pi, in [-pi, pi)
                const float vz = fmaf(cp, f.az, fmaf(sp, f.bz, f.cz));
                if (vz < 0.0f) {
                    // a4: ground = G + (sd / v_z) N,  N = cos' P + sin' Q
                    const float rho = sd * rcp_approx(vz);
                    const float gx = fmaf(rho, fmaf(cp, f.px, sp * f.qx), f.gx);
                    const float gy = fmaf(rho, fmaf(cp, f.py, sp * f.qy), f.gy);
                    float vx = 0.0f, vy = 0.0f;
                    if (!COPLANAR) {
                        const float *fr = &sm.frame[e * kFrameStride];
                        vx = fmaf(cp, fr[F_AX], fmaf(sp, fr[F_BX], fr[F_CX]));
                        vy = fmaf(cp, fr[F_AY], fmaf(sp, fr[F_BY], fr[F_CY]));
                    }
                    cm = plane_candidates<TELSRC, COPLANAR, NT, REFR>(P, gx, gy, vx, vy, vz, &cell);
                } else {
                    ++n_up;
                }
            } else {
                // the same hoisted Philox as the axis kind (the process tag is counter word 3)
                r = kind_tag(kind) ? philox_photon(P, pe, j, 1u) : cherenkov_words(philox_photon(P, pe, j >> 1, 0u), j);
                bool up;
                if (!polar_cull(sm, e, kind, r.r3, &up))
                    cm = generic_candidates<TELSRC, COPLANAR, NT, REFR>(P, sm, e, r.r0, r.r1, r.r2, r.r3, &cell, &up);
                if (up) ++n_up;
            }
        }
        if constexpr (tel_base(TELSRC) == TEL_CONST) {
            if (cm == kAllTelescopes) cm = (1u << NT) - 1u;          // flat photon: all slots go to the exact test
        } else {
            const uint32_t wide = __ballot_sync(0xffffffffu, cm == kAllTelescopes);
            if (wide) {
                wide_push<TELSRC, MODE>(P, sm, tile_first, q_head, q_count, wide, e, j);
                if (cm == kAllTelescopes) cm = 0u;
            }
        }
        const uint32_t have = __ballot_sync(0xffffffffu, cm != 0u);
        if (__popc(have) >= kDenseMin) {
            // dense iteration: each lane's first candidate is evaluated on the spot, further ones are queued
            const bool has = cm != 0u;
            int k = 0;
            if (has) { k = (int)slot_telescope<TELSRC>(cell, __ffs(cm) - 1); cm &= cm - 1u; }
            dense_eval<TELSRC, MODE>(P, sm, tile_first, e, j, r.r0, r.r1, r.r2, r.r3, k, has);
        }
        if (__any_sync(0xffffffffu, cm != 0u))
            push_candidates<TELSRC, MODE>(P, sm, tile_first, q_head, q_count, cm, e, j, [&](int c) { return slot_telescope<TELSRC>(cell, c); });
    }
    ww.e = e; ww.kind = kind; ww.end = end; ww.g = g; ww.j = j; ww.n_up = n_up; ww.q_head = q_head; ww.q_count = q_count;
    ww.pe = pe; ww.f_reg = f_reg;
}

// The pair loop (tally kernels, ground histogram, and the sparse tiles of the photon-output kernels): a lane takes the two
// adjacent slots g, g + 1 (g even) of the index space per trip, a warp 64.  Both photons belong to the same emitter
// (the index space is padded to even counts), so one emitter state serves both; their Philox chains and geometry are
// independent and interleave, which halves the dependent-issue stalls per photon, and the round keys / telescope
// constants are fetched once for two photons.  Walks the warp's photons [base, hi), base even.
// FULL: [base, hi) is a whole number of trips (no lane ever runs past hi).
template <int TELSRC, bool COPLANAR, int NT, int MODE, bool REFR, bool INLINE, bool FULL = false>
__device__ __forceinline__ void walk_pairs(const KParams &P, TileSmem &sm, const uint32_t base, const uint32_t hi,
                                           const unsigned long long tile_first, uint32_t &n_up_out, uint32_t &q_head, uint32_t &q_count)
{
    constexpr bool kFrameInRegs = (tel_base(TELSRC) == TEL_CONST);
    const int lane = threadIdx.x & 31;
    if (base >= hi) return;
    uint32_t g = base + 2u * (uint32_t)lane;
    int e;
    {
        const uint32_t g0 = min(g, hi - 2u);
        int a = 0, b = kTile;                 // invariant: prefix[a] <= g0 < prefix[b]
        while (b - a > 1) { const int m = (a + b) >> 1; if (sm.prefix[m] <= g0) a = m; else b = m; }
        e = a;
    }
    uint32_t end = sm.prefix[e + 1], rend = end - sm.odd[e], j = g - sm.prefix[e], n_up = 0u;
    int kind = sm.kind[e];
    // brute-force kernels: the telescopes this lane's emitter can reach; bit 8 = not the axis kind (its candidates do
    // not come from the pre-tests below)
    uint32_t reach = (uint32_t)sm.tmask[e] | ((kind != KIND_CHER_AXIS) ? 0x100u : 0u);
    PhiloxEmitter pe = philox_emitter(P, emitter_segment(P, tile_first, e));
    AxisFrame f_reg = load_axis_frame(sm, e);
    for (uint32_t b0 = base; b0 < hi; b0 += 64u, g += 64u, j += 64u) {
        const bool active = FULL || g < hi;
        // brute-force kernels: the telescopes that any lane's emitter can reach at all (reach_mask); the pre-tests of the
        // others are skipped for the whole warp (most emitters of a shower reach none; a trip spans one or two emitters)
        uint32_t umask = 0xffu;
        if constexpr (tel_base(TELSRC) == TEL_CONST) {
            if (active && g >= end) {
                do { ++e; end = sm.prefix[e + 1]; } while (g >= end);
                rend = end - sm.odd[e];
                j = g - sm.prefix[e];
                kind = sm.kind[e];
                reach = (uint32_t)sm.tmask[e] | ((kind != KIND_CHER_AXIS) ? 0x100u : 0u);
                pe = philox_emitter(P, emitter_segment(P, tile_first, e));
                f_reg = load_axis_frame(sm, e);
            }
            umask = __reduce_or_sync(0xffffffffu, active ? reach : 0u);
        }
        uint32_t cmA = 0u, cmB = 0u;
        uint2 cellA = make_uint2(0xffffffffu, 0xffffffffu), cellB = cellA;
        Rand4 rA = {0u, 0u, 0u, 0u}, rB = rA;
        Hit hA, hB;                                   // INLINE (ground histogram): both photons evaluated on the spot
        hA.ok = false; hA.k = 0; hA.x = hA.y = hA.vx = hA.vy = hA.t = hA.lam = hA.w = 0.0f;
        hB = hA;
        if (active) {
            if (tel_base(TELSRC) != TEL_CONST && g >= end) {
                do { ++e; end = sm.prefix[e + 1]; } while (g >= end);
                rend = end - sm.odd[e];
                j = g - sm.prefix[e];
                kind = sm.kind[e];
                pe = philox_emitter(P, emitter_segment(P, tile_first, e));
                if (kFrameInRegs) f_reg = load_axis_frame(sm, e);
            }
            const bool hasB = g + 1u < rend;                     // slot g + 1 is empty after an odd count
            if (kind == KIND_CHER_AXIS) {
                const AxisFrame f = kFrameInRegs ? f_reg : load_axis_frame(sm, e);
                const Rand4 blk = philox_photon(P, pe, j >> 1, 0u);                               // a2: one block, two photons (R20; j is even)
                rA = Rand4{blk.r0, blk.r1, 0u, 0u};
                rB = Rand4{blk.r2, blk.r3, 0u, 0u};
                // a3 / a4 as in walk(), for both photons
                const float sdA = fmaf(one_two(rA.r0), f.negL, f.k0c), sdB = fmaf(one_two(rB.r0), f.negL, f.k0c);
                float spA, cpA, spB, cpB;
                __sincosf(fmaf(one_two(rA.r1), 6.2831853f, -9.42477760f), &spA, &cpA);
                __sincosf(fmaf(one_two(rB.r1), 6.2831853f, -9.42477760f), &spB, &cpB);
                const float vzA = fmaf(cpA, f.az, fmaf(spA, f.bz, f.cz)), vzB = fmaf(cpB, f.az, fmaf(spB, f.bz, f.cz));
                // the crossing of the reference plane and (non-coplanar arrays) the horizontal direction: only where a
                // telescope is in reach of the warp (brute-force kernels: umask; a shower's light mostly reaches none)
                float gxA = 0.0f, gyA = 0.0f, gxB = 0.0f, gyB = 0.0f, vxA = 0.0f, vyA = 0.0f, vxB = 0.0f, vyB = 0.0f;
                if (tel_base(TELSRC) != TEL_CONST || umask != 0u) {
                    const float rhoA = sdA * rcp_approx(vzA), rhoB = sdB * rcp_approx(vzB);
                    gxA = fmaf(rhoA, fmaf(cpA, f.px, spA * f.qx), f.gx); gyA = fmaf(rhoA, fmaf(cpA, f.py, spA * f.qy), f.gy);
                    gxB = fmaf(rhoB, fmaf(cpB, f.px, spB * f.qx), f.gx); gyB = fmaf(rhoB, fmaf(cpB, f.py, spB * f.qy), f.gy);
                    if (!COPLANAR) {
                        const float *fr = &sm.frame[e * kFrameStride];
                        vxA = fmaf(cpA, fr[F_AX], fmaf(spA, fr[F_BX], fr[F_CX])); vyA = fmaf(cpA, fr[F_AY], fmaf(spA, fr[F_BY], fr[F_CY]));
                        vxB = fmaf(cpB, fr[F_AX], fmaf(spB, fr[F_BX], fr[F_CX])); vyB = fmaf(cpB, fr[F_AY], fmaf(spB, fr[F_BY], fr[F_CY]));
                    }
                }
                if constexpr (tel_base(TELSRC) == TEL_CONST) {
                    // the pre-tests of both photons, telescope by telescope, for the telescopes in reach of the warp
                    const bool dnA = vzA < 0.0f, dnB = hasB && vzB < 0.0f;
                    n_up += (dnA ? 0u : 1u) + ((hasB && !dnB) ? 1u : 0u);
                    if (umask != 0u) {
                        const float vz2sA = vzA * vzA * 0.9999f, vz2sB = vzB * vzB * 0.9999f;
                        const float addA = REFR ? refraction_slack(P, vzA) : 0.0f, addB = REFR ? refraction_slack(P, vzB) : 0.0f;
#pragma unroll
                        for (int k = 0; k < NT; ++k) {
                            if ((umask >> k) & 1u) {
                                if (dnA && plane_pretest<COPLANAR>(P.tel_c[k], gxA, gyA, vxA, vyA, vzA, vz2sA, addA)) cmA |= 1u << k;
                                if (dnB && plane_pretest<COPLANAR>(P.tel_c[k], gxB, gyB, vxB, vyB, vzB, vz2sB, addB)) cmB |= 1u << k;
                            }
                        }
                    }
                } else {
                    if (vzA < 0.0f) cmA = plane_candidates<TELSRC, COPLANAR, NT, REFR>(P, gxA, gyA, vxA, vyA, vzA, &cellA); else ++n_up;
                    if (hasB) {
                        if (vzB < 0.0f) cmB = plane_candidates<TELSRC, COPLANAR, NT, REFR>(P, gxB, gyB, vxB, vyB, vzB, &cellB); else ++n_up;
                    }
                }
                if constexpr (INLINE) {
                    const float *fr = &sm.frame[e * kFrameStride];
                    if (cmA != 0u && cmA != kAllTelescopes) {
                        Photon ph;
                        ph.axis = true; ph.tag = 0; ph.u3 = cherenkov_u3(rA.r0, rA.r1);
                        ph.vx = fmaf(cpA, fr[F_AX], fmaf(spA, fr[F_BX], fr[F_CX])); ph.vy = fmaf(cpA, fr[F_AY], fmaf(spA, fr[F_BY], fr[F_CY]));
                        ph.vz = vzA; ph.gx = gxA; ph.gy = gyA; ph.s = (one_two(rA.r0) - kOneMinus) * fr[F_LEN]; ph.ez = -sdA * fr[F_DZ];
                        ph.ex = ph.ey = 0.0f; ph.rva = rcp_approx(vzA);
                        const int k = (int)slot_telescope<TELSRC>(cellA, __ffs(cmA) - 1);
                        cmA &= cmA - 1u;
                        hA = evaluate_pair<TELSRC, COPLANAR>(P, sm, e, ph, k);
                    }
                    if (cmB != 0u && cmB != kAllTelescopes) {
                        Photon ph;
                        ph.axis = true; ph.tag = 0; ph.u3 = cherenkov_u3(rB.r0, rB.r1);
                        ph.vx = fmaf(cpB, fr[F_AX], fmaf(spB, fr[F_BX], fr[F_CX])); ph.vy = fmaf(cpB, fr[F_AY], fmaf(spB, fr[F_BY], fr[F_CY]));
                        ph.vz = vzB; ph.gx = gxB; ph.gy = gyB; ph.s = (one_two(rB.r0) - kOneMinus) * fr[F_LEN]; ph.ez = -sdB * fr[F_DZ];
                        ph.ex = ph.ey = 0.0f; ph.rva = rcp_approx(vzB);
                        const int k = (int)slot_telescope<TELSRC>(cellB, __ffs(cmB) - 1);
                        cmB &= cmB - 1u;
                        hB = evaluate_pair<TELSRC, COPLANAR>(P, sm, e, ph, k);
                    }
                }
            } else {
                const uint32_t tag = kind_tag(kind);
                bool up;
                const Rand4 blk0 = philox_photon(P, pe, tag ? j : (j >> 1), tag);
                rA = tag ? blk0 : Rand4{blk0.r0, blk0.r1, 0u, 0u};
                if (!polar_cull(sm, e, kind, rA.r3, &up))
                    cmA = generic_candidates<TELSRC, COPLANAR, NT, REFR>(P, sm, e, rA.r0, rA.r1, rA.r2, rA.r3, &cellA, &up);
                if (up) ++n_up;
                if (hasB) {
                    rB = tag ? philox_photon(P, pe, j + 1u, 1u) : Rand4{blk0.r2, blk0.r3, 0u, 0u};
                    if (!polar_cull(sm, e, kind, rB.r3, &up))
                        cmB = generic_candidates<TELSRC, COPLANAR, NT, REFR>(P, sm, e, rB.r0, rB.r1, rB.r2, rB.r3, &cellB, &up);
                    if (up) ++n_up;
                }
            }
        }
        if constexpr (INLINE) {
            const unsigned long long id0 = (emitter_segment(P, tile_first, e) << 25) | (unsigned long long)j;
            commit_hits<MODE>(P, sm, hA, id0);
            commit_hits<MODE>(P, sm, hB, id0 + 1ull);
        }
        // candidates of slot A, then of slot B: wide test / on-the-spot evaluation / queue, as in walk()
        // (most trips of a shower's light hold none: one vote skips the lot)
        // (photon output: nothing in reach of the warp = no candidate, without the vote; the tally kernels, whose dispatch
        // below is one test, measured slower with this branch: c2 0.678 -> 0.685 ms, c5 7.21 -> 7.01 ms)
        if constexpr (tel_base(TELSRC) == TEL_CONST && MODE != MODE_TALLY) { if (umask == 0u) continue; }
        if (!__any_sync(0xffffffffu, (cmA | cmB) != 0u)) continue;
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            uint32_t cm = s ? cmB : cmA;
            const uint2 cell = s ? cellB : cellA;
            const Rand4 r = s ? rB : rA;
            const uint32_t jj = j + (uint32_t)s;
            if constexpr (tel_base(TELSRC) == TEL_CONST) {
                if (cm == kAllTelescopes) cm = (1u << NT) - 1u;
            } else {
                const uint32_t wide = __ballot_sync(0xffffffffu, cm == kAllTelescopes);
                if (wide) {
                    wide_push<TELSRC, MODE>(P, sm, tile_first, q_head, q_count, wide, e, jj);
                    if (cm == kAllTelescopes) cm = 0u;
                }
            }
            const uint32_t have = __ballot_sync(0xffffffffu, cm != 0u);
            if constexpr (MODE != MODE_TALLY) {
                if (__popc(have) >= kDenseMin) {
                    const bool has = cm != 0u;
                    int k = 0;
                    if (has) { k = (int)slot_telescope<TELSRC>(cell, __ffs(cm) - 1); cm &= cm - 1u; }
                    dense_eval<TELSRC, MODE>(P, sm, tile_first, e, jj, r.r0, r.r1, r.r2, r.r3, k, has);
                }
                if (__any_sync(0xffffffffu, cm != 0u))
                    push_candidates<TELSRC, MODE>(P, sm, tile_first, q_head, q_count, cm, e, jj, [&](int c) { return slot_telescope<TELSRC>(cell, c); });
            } else {
                if (have)
                    push_candidates<TELSRC, MODE>(P, sm, tile_first, q_head, q_count, cm, e, jj, [&](int c) { return slot_telescope<TELSRC>(cell, c); });
            }
        }
    }
    n_up_out += n_up;
}

// Dense tiles, generic kinds (and the probe): a3 + a4 of one photon out of line -- photon in the global frame, the
// conservative pre-tests over the NT constant-bank telescopes, the exact test of the first candidate.  *cm_left = the
// further candidates (bit k = telescope k), *upward = the photon does not go down.
template <bool COPLANAR, int NT, bool REFR>
__device__ __forceinline__ uint32_t const_candidates(const KParams &P, const Photon &ph)
{
    if (ph.vz > -0.05f) return (1u << NT) - 1u;                      // flat photon: every slot goes to the exact test
    uint2 cell;
    if (ph.axis) return plane_candidates<TEL_CONST, COPLANAR, NT, REFR>(P, ph.gx, ph.gy, ph.vx, ph.vy, ph.vz, &cell);
    const float spl = -ph.ez * rcp_approx(ph.vz);                    // candidate search only: the pre-tests carry slack
    return plane_candidates<TEL_CONST, COPLANAR, NT, REFR>(P, fmaf(spl, ph.vx, ph.ex), fmaf(spl, ph.vy, ph.ey), ph.vx, ph.vy, ph.vz, &cell);
}

struct GenericHit { Hit h; uint32_t cm_left; bool upward; };

template <bool COPLANAR, int NT, bool REFR>
__device__ __noinline__ GenericHit generic_hit(const KParams &P, TileSmem &sm, int e, const Rand4 r, uint32_t j)
{
    GenericHit g;
    g.h.ok = false; g.h.k = 0; g.h.x = g.h.y = g.h.vx = g.h.vy = g.h.t = g.h.lam = g.h.w = 0.0f;
    g.cm_left = 0u;
    const Photon ph = photon_from_rand(P, sm, e, r);
    g.upward = !(ph.vz < 0.0f);
    if (g.upward) return g;
    uint32_t cm = const_candidates<COPLANAR, NT, REFR>(P, ph);
    if (cm != 0u) {
        const int k = __ffs(cm) - 1;
        cm &= cm - 1u;
        g.h = evaluate_any<TEL_CONST, COPLANAR>(P, sm, e, ph, k, j);
    }
    g.cm_left = cm;
    return g;
}

// ------------------------------------------------------------------------------------
// Photon output, brute-force kernels: is this tile dense (a good part of its photons hit one telescope: c5g, a detector
// that covers the light pool) or sparse (c5: 0.4 % hit)?  Every lane takes one photon of its warp's range, evenly
// spread over it (even slots always hold a photon), draws it and runs the conservative pre-test only; the candidates
// are counted per telescope in os.probe.  Nothing is tallied or written: the loops start from the beginning afterwards.
template <bool COPLANAR, int NT, bool REFR>
__device__ __noinline__ void probe_density(const KParams &P, TileSmem &sm, OutSmem &os, const uint32_t lo, const uint32_t hi,
                                           const unsigned long long tile_first)
{
    const uint32_t lane = lane_id();
    uint32_t cm = 0u;
    if (lo < hi) {
        const uint32_t stride = max(2u, ((hi - lo) >> 5) & ~1u), g = lo + stride * lane;
        if (g < hi) {
            int a = 0, b = kTile;                 // invariant: prefix[a] <= g < prefix[b]
            while (b - a > 1) { const int m = (a + b) >> 1; if (sm.prefix[m] <= g) a = m; else b = m; }
            const int e = a;
            const uint32_t j = g - sm.prefix[e];
            const unsigned long long S = emitter_segment(P, tile_first, e);
            const uint32_t tag = kind_tag(sm.kind[e]);
            const Rand4 blk = philox4x32_10(P, tag ? j : (j >> 1), (uint32_t)S, (uint32_t)(S >> 32), tag);
            const Rand4 r = tag ? blk : cherenkov_words(blk, j);
            const Photon ph = photon_from_rand(P, sm, e, r);
            if (ph.vz <= -0.05f) cm = const_candidates<COPLANAR, NT, REFR>(P, ph);
        }
    }
#pragma unroll
    for (int k = 0; k < NT; ++k) {
        const uint32_t c = (uint32_t)__popc(__ballot_sync(0xffffffffu, (cm >> k) & 1u));
        if (c && lane == 0u) atomicAdd(&os.probe[k], c);
    }
}

// The photon loop of a dense tile (photon output, brute-force kernels).  The pair loop of walk_pairs -- a lane takes
// the adjacent slots g, g + 1 per trip, one Philox block for both (R20) -- with every candidate evaluated on the spot
// from the values in registers, the records of a round (SUB trips, <= 64 SUB records) staged per warp and their slots
// reserved once per tile and round (OutSmem).  Per round r:  pick up the base of round r - 2 and copy that block out
// (copy_block)  ->  arithmetic of round r, staged into the buffer that block left  ->  arrive at round r.  The global
// atomic of a round, its latency and the spread between the warps of the tile are thus covered by a round of
// arithmetic, and there is no block barrier.  Every warp of the tile runs all the rounds (it arrives with 0 records
// once its range is finished).
// kd = the tile's dense telescope; hits on other telescopes, further candidates of a photon and the generic kinds
// take the paths of the sparse loop (queue / direct cursor bump).
// FAST: one coplanar telescope, no refraction corrections, no transmission table, no id side buffer (the launch that
// is measured against the HBM roofline): the exact evaluation of an axis-kind photon written out on the values the
// loop holds, built from the same pieces as evaluate_pair (bit-identical records), two trips per round.
template <bool COPLANAR, int NT, bool REFR, bool FAST>
__device__ __forceinline__ void walk_dense(const KParams &P, TileSmem &sm, OutSmem &os, const uint32_t base, const uint32_t hi,
                                           const unsigned long long tile_first, const uint32_t n_trips, const int kd,
                                           uint32_t &n_up_out, uint32_t &q_head, uint32_t &q_count)
{
    constexpr int TELSRC = TEL_CONST;
    constexpr uint32_t SUB = FAST ? (uint32_t)kFastSub : 1u, NB = FAST ? (uint32_t)kFastBufs : 2u;
    constexpr uint32_t kBufWords = (uint32_t)kWarpStageWords / NB;
    static_assert(!FAST || (NT == 1 && COPLANAR && !REFR), "fast path: one coplanar telescope, straight lines");
    const uint32_t lane = lane_id(), warp = threadIdx.x >> 5, lt = (1u << lane) - 1u;
    const bool want_ids = !FAST && P.ids != nullptr;
    const unsigned long long cap_kd = P.tel_capacity[kd], off_kd = P.tel_offset[kd];
    uint32_t g = base + 2u * lane;
    int e;
    {
        const uint32_t g0 = (base < hi) ? min(g, hi - 2u) : 0u;
        int a = 0, b = kTile;                 // invariant: prefix[a] <= g0 < prefix[b]
        while (b - a > 1) { const int m = (a + b) >> 1; if (sm.prefix[m] <= g0) a = m; else b = m; }
        e = a;
    }
    uint32_t end = sm.prefix[e + 1], rend = end - sm.odd[e], j = g - sm.prefix[e], n_up = 0u;
    int kind = sm.kind[e];
    PhiloxEmitter pe = philox_emitter(P, emitter_segment(P, tile_first, e));
    AxisFrame f = load_axis_frame(sm, e);
    uint32_t n_h[NB], off_h[NB];                    // the blocks staged 1 .. NB rounds ago: records, offset in their round
#pragma unroll
    for (uint32_t i = 0; i < NB; ++i) { n_h[i] = 0u; off_h[i] = 0u; }
    // this thread's tally of hits on kd: fp32 partial sums over kTallyRounds rounds (<= 4 kTallyRounds terms), then fp64
    constexpr uint32_t kTallyRounds = 16u;
    uint32_t acc_n = 0u;
    float part_w = 0.0f, part_wt = 0.0f;
    double acc_w = 0.0, acc_wt = 0.0;
    const uint32_t n_rounds = (n_trips + SUB - 1u) / SUB;
    // The warp that arrives last at a round bumps the cursor, but does not wait for the answer (2-3 us under the write
    // load): it publishes the base only after the arithmetic of its next trip (lane 0: pend_b is the pending result).
    unsigned long long pend_b = 0ull;
    uint32_t pend_r = 0xffffffffu;
    auto publish_pending = [&]() {
        if (lane == 0u && pend_r != 0xffffffffu) {
            *(volatile unsigned long long *)&os.rbase[pend_r & (kRoundSlots - 1)] = pend_b;
            mbar_arrive_release(&os.rbar[pend_r & (kRoundSlots - 1)]);
            pend_r = 0xffffffffu;
        }
    };
    for (uint32_t r = 0; r < n_rounds; ++r) {
        float *const st = os.stage[warp] + (r % NB) * kBufWords;
        unsigned long long *const sid = reinterpret_cast<unsigned long long *>(st + kBlockRecs * kRecWords);
        // the block staged NB rounds ago leaves this buffer (its slots have been reserved meanwhile)
        if (r >= NB) {
            if (want_ids) copy_block<SUB, true>(P, os, st, cap_kd, off_kd, n_h[NB - 1], off_h[NB - 1], r - NB);
            else copy_block<SUB, false>(P, os, st, cap_kd, off_kd, n_h[NB - 1], off_h[NB - 1], r - NB);
        }
        __syncwarp();
        uint32_t cnt = 0u;                           // records staged in this round (warp-uniform)
#pragma unroll
        for (uint32_t t = 0; t < SUB; ++t, g += 64u, j += 64u) {
            const bool active = g < hi;
            uint32_t cmA = 0u, cmB = 0u;
            Hit hA, hB;
            hA.ok = false; hB.ok = false;
            if (active) {
                if (g >= end) {
                    do { ++e; end = sm.prefix[e + 1]; } while (g >= end);
                    rend = end - sm.odd[e];
                    j = g - sm.prefix[e];
                    kind = sm.kind[e];
                    pe = philox_emitter(P, emitter_segment(P, tile_first, e));
                    f = load_axis_frame(sm, e);
                }
                const bool hasB = g + 1u < rend;                     // slot g + 1 is empty after an odd count
                if (kind == KIND_CHER_AXIS) {
                    const Rand4 blk = philox_photon(P, pe, j >> 1, 0u);                               // a2: one block, two photons (R20; j is even)
                    // a3 / a4 as in walk_pairs, for both photons
                    const float w1A = one_two(blk.r0), w1B = one_two(blk.r2);
                    const float sdA = fmaf(w1A, f.negL, f.k0c), sdB = fmaf(w1B, f.negL, f.k0c);
                    float spA, cpA, spB, cpB;
                    __sincosf(fmaf(one_two(blk.r1), 6.2831853f, -9.42477760f), &spA, &cpA);
                    __sincosf(fmaf(one_two(blk.r3), 6.2831853f, -9.42477760f), &spB, &cpB);
                    const float vzA = fmaf(cpA, f.az, fmaf(spA, f.bz, f.cz)), vzB = fmaf(cpB, f.az, fmaf(spB, f.bz, f.cz));
                    const float rvA = rcp_approx(vzA), rvB = rcp_approx(vzB);
                    const float rhoA = sdA * rvA, rhoB = sdB * rvB;
                    const float gxA = fmaf(rhoA, fmaf(cpA, f.px, spA * f.qx), f.gx), gyA = fmaf(rhoA, fmaf(cpA, f.py, spA * f.qy), f.gy);
                    const float gxB = fmaf(rhoB, fmaf(cpB, f.px, spB * f.qx), f.gx), gyB = fmaf(rhoB, fmaf(cpB, f.py, spB * f.qy), f.gy);
                    const float *fr = &sm.frame[e * kFrameStride];
                    const float4 vc0 = *reinterpret_cast<const float4 *>(fr + F_AX);      // AX, AY, BX, BY
                    const float4 vc1 = *reinterpret_cast<const float4 *>(fr + F_CX);      // CX, CY, LEN, LAYER
                    const float4 hs = *reinterpret_cast<const float4 *>(fr + F_W0);       // W0, T0, IBC, DZ
                    const float vxA = fmaf(cpA, vc0.x, fmaf(spA, vc0.z, vc1.x)), vyA = fmaf(cpA, vc0.y, fmaf(spA, vc0.w, vc1.y));
                    const float vxB = fmaf(cpB, vc0.x, fmaf(spB, vc0.z, vc1.x)), vyB = fmaf(cpB, vc0.y, fmaf(spB, vc0.w, vc1.y));
                    if constexpr (FAST) {
                        // evaluate_pair<TEL_CONST, true> for telescope 0, straight lines, no transmission table
                        const float4 T = P.tel_c[0];
                        const float telT = P.telT_c[0];
                        const int li_frame = __float_as_int(vc1.w);
                        const float h_next = fr[F_HNEXT];
                        {
                            const float rv = fmaf(rvA, fmaf(-vzA, rvA, 1.0f), rvA), ez = -sdA * hs.w;
                            float s_pl;
                            hA.x = gxA - T.x; hA.y = gyA - T.y;
                            const bool ok = axis_test_coplanar(hA.x, hA.y, vxA, vyA, ez, rv, T.w, &s_pl);
                            if (!(vzA < 0.0f)) ++n_up;
                            hA.ok = ok && (vzA < 0.0f);
                            const float habs = P.z_ref_f + ez;
                            float E;
                            const float Te = depth_at(P.layerf[emission_layer(P, li_frame, h_next, habs)], habs, &E);
                            hA.t = arrival_time(P, (w1A - kOneMinus) * vc1.z, hs.z, hs.y, s_pl, telT, Te, rv);
                            hA.lam = cherenkov_lambda(P, cherenkov_u3(blk.r0, blk.r1));
                            hA.vx = vxA; hA.vy = vyA; hA.w = hs.x;
                        }
                        if (hasB) {
                            const float rv = fmaf(rvB, fmaf(-vzB, rvB, 1.0f), rvB), ez = -sdB * hs.w;
                            float s_pl;
                            hB.x = gxB - T.x; hB.y = gyB - T.y;
                            const bool ok = axis_test_coplanar(hB.x, hB.y, vxB, vyB, ez, rv, T.w, &s_pl);
                            if (!(vzB < 0.0f)) ++n_up;
                            hB.ok = ok && (vzB < 0.0f);
                            const float habs = P.z_ref_f + ez;
                            float E;
                            const float Te = depth_at(P.layerf[emission_layer(P, li_frame, h_next, habs)], habs, &E);
                            hB.t = arrival_time(P, (w1B - kOneMinus) * vc1.z, hs.z, hs.y, s_pl, telT, Te, rv);
                            hB.lam = cherenkov_lambda(P, cherenkov_u3(blk.r2, blk.r3));
                            hB.vx = vxB; hB.vy = vyB; hB.w = hs.x;
                        }
                    } else {
                        // one telescope: the exact test decides; several: the conservative pre-tests pick the candidates
                        uint2 cell;
                        if (vzA < 0.0f) cmA = (NT == 1) ? 1u : plane_candidates<TELSRC, COPLANAR, NT, REFR>(P, gxA, gyA, vxA, vyA, vzA, &cell); else ++n_up;
                        if (hasB) {
                            if (vzB < 0.0f) cmB = (NT == 1) ? 1u : plane_candidates<TELSRC, COPLANAR, NT, REFR>(P, gxB, gyB, vxB, vyB, vzB, &cell); else ++n_up;
                        }
                        if (cmA != 0u) {
                            Photon ph;
                            ph.axis = true; ph.tag = 0; ph.u3 = cherenkov_u3(blk.r0, blk.r1);
                            ph.vx = vxA; ph.vy = vyA; ph.vz = vzA; ph.gx = gxA; ph.gy = gyA; ph.rva = rvA;
                            ph.s = (w1A - kOneMinus) * vc1.z; ph.ez = -sdA * hs.w;
                            ph.ex = ph.ey = 0.0f;
                            const int k = (NT == 1) ? 0 : __ffs(cmA) - 1;
                            cmA &= cmA - 1u;
                            hA = evaluate_pair<TELSRC, COPLANAR>(P, sm, e, ph, k);
                        }
                        if (cmB != 0u) {
                            Photon ph;
                            ph.axis = true; ph.tag = 0; ph.u3 = cherenkov_u3(blk.r2, blk.r3);
                            ph.vx = vxB; ph.vy = vyB; ph.vz = vzB; ph.gx = gxB; ph.gy = gyB; ph.rva = rvB;
                            ph.s = (w1B - kOneMinus) * vc1.z; ph.ez = -sdB * hs.w;
                            ph.ex = ph.ey = 0.0f;
                            const int k = (NT == 1) ? 0 : __ffs(cmB) - 1;
                            cmB &= cmB - 1u;
                            hB = evaluate_pair<TELSRC, COPLANAR>(P, sm, e, ph, k);
                        }
                    }
                } else {
                    // generic kinds: out of line (photon in the global frame, pre-tests, exact test of the first candidate)
                    const uint32_t tag = kind_tag(kind);
                    const Rand4 blk0 = philox_photon(P, pe, tag ? j : (j >> 1), tag);
                    bool up;
                    if (!polar_cull(sm, e, kind, blk0.r3, &up)) {
                        const GenericHit ga = generic_hit<COPLANAR, NT, REFR>(P, sm, e, tag ? blk0 : Rand4{blk0.r0, blk0.r1, 0u, 0u}, j);
                        hA = ga.h; cmA = ga.cm_left; up = ga.upward;
                    }
                    if (up) ++n_up;
                    if (hasB) {
                        const Rand4 rB = tag ? philox_photon(P, pe, j + 1u, 1u) : Rand4{blk0.r2, blk0.r3, 0u, 0u};
                        if (!polar_cull(sm, e, kind, rB.r3, &up)) {
                            const GenericHit gb = generic_hit<COPLANAR, NT, REFR>(P, sm, e, rB, j + 1u);
                            hB = gb.h; cmB = gb.cm_left; up = gb.upward;
                        }
                        if (up) ++n_up;
                    }
                }
            }
            unsigned long long idA = 0ull;
            if (want_ids) idA = (emitter_segment(P, tile_first, e) << 25) | ((unsigned long long)kind_tag(kind) << 24) | (unsigned long long)j;
            bool sA = hA.ok, sB = hB.ok;
            if constexpr (NT > 1) {
                // hits on another telescope than the tile's dense one: tallied and written directly
                const bool oA = hA.ok && hA.k != kd, oB = hB.ok && hB.k != kd;
                if (__any_sync(0xffffffffu, oA || oB)) {
                    if (!want_ids) idA = (emitter_segment(P, tile_first, e) << 25) | ((unsigned long long)kind_tag(kind) << 24) | (unsigned long long)j;
                    Hit h2 = hA; h2.ok = oA;
                    commit_hits<MODE_OUT>(P, sm, h2, idA);
                    h2 = hB; h2.ok = oB;
                    commit_hits<MODE_OUT>(P, sm, h2, idA + 1ull);
                }
                sA = hA.ok && !oA; sB = hB.ok && !oB;
            }
            if constexpr (!FAST) {
                // further candidates of the two photons (several telescopes; flat photons of the generic kinds): queue
                if (__any_sync(0xffffffffu, (cmA | cmB) != 0u)) {
                    push_candidates<TELSRC, MODE_OUT>(P, sm, tile_first, q_head, q_count, cmA, e, j, [&](int c) { return (uint32_t)c; });
                    push_candidates<TELSRC, MODE_OUT>(P, sm, tile_first, q_head, q_count, cmB, e, j + 1u, [&](int c) { return (uint32_t)c; });
                }
            }
            {
                // (a miss leaves t undefined: select the product, not the factor)
                const float wA = sA ? hA.w : 0.0f, wB = sB ? hB.w : 0.0f;
                part_w += wA + wB;
                part_wt += (sA ? hA.w * hA.t : 0.0f) + (sB ? hB.w * hB.t : 0.0f);
            }
            const uint32_t mA = __ballot_sync(0xffffffffu, sA), mB = __ballot_sync(0xffffffffu, sB);
            const uint32_t nA = (uint32_t)__popc(mA);
            if (sA) {
                const uint32_t s = cnt + (uint32_t)__popc(mA & lt);
                float *rec = st + s * kRecWords;
                rec[0] = hA.x; rec[1] = hA.y; rec[2] = hA.vx; rec[3] = hA.vy; rec[4] = hA.t; rec[5] = hA.lam; rec[6] = hA.w;
                if (want_ids) sid[s] = idA;
            }
            if (sB) {
                const uint32_t s = cnt + nA + (uint32_t)__popc(mB & lt);
                float *rec = st + s * kRecWords;
                rec[0] = hB.x; rec[1] = hB.y; rec[2] = hB.vx; rec[3] = hB.vy; rec[4] = hB.t; rec[5] = hB.lam; rec[6] = hB.w;
                if (want_ids) sid[s] = idA + 1ull;
            }
            cnt += nA + (uint32_t)__popc(mB);
            if (t == 0u) publish_pending();
        }
        acc_n += cnt;                               // warp-uniform: lane 0's copy is the one that counts
        if ((r & (kTallyRounds - 1u)) == kTallyRounds - 1u) { acc_w += (double)part_w; acc_wt += (double)part_wt; part_w = 0.0f; part_wt = 0.0f; }
        __syncwarp();
        uint32_t old = 0u;
        if (lane == 0u) {
            old = add_acq_rel_cta(&os.agg[r & (kRoundSlots - 1)], (cnt << 8) | 1u);
            if ((old & 0xffu) == (uint32_t)kWarps - 1u) {
                // last arrival of round r: reserve the round's records, publish the base
                const uint32_t total = (old >> 8) + cnt;
                os.agg[r & (kRoundSlots - 1)] = 0u;
                pend_b = 0ull;
                if (total) pend_b = atomicAdd(&P.cursors[kd], (unsigned long long)total);
                pend_r = r;
            }
        }
        __syncwarp();
#pragma unroll
        for (uint32_t i = NB - 1u; i > 0u; --i) { n_h[i] = n_h[i - 1u]; off_h[i] = off_h[i - 1u]; }
        off_h[0] = __shfl_sync(0xffffffffu, old >> 8, 0);
        n_h[0] = cnt;
    }
    publish_pending();
    // the last NB blocks, oldest first
#pragma unroll
    for (uint32_t i = NB; i > 0u; --i) {
        if (n_rounds >= i) {
            const uint32_t r = n_rounds - i;
            const float *st = os.stage[warp] + (r % NB) * kBufWords;
            if (want_ids) copy_block<SUB, true>(P, os, st, cap_kd, off_kd, n_h[i - 1u], off_h[i - 1u], r);
            else copy_block<SUB, false>(P, os, st, cap_kd, off_kd, n_h[i - 1u], off_h[i - 1u], r);
        }
    }
    // the warp's tally of kd into the tile's: one shared-memory atomic per warp and sum
    acc_w += (double)part_w; acc_wt += (double)part_wt;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { acc_w += __shfl_xor_sync(0xffffffffu, acc_w, o); acc_wt += __shfl_xor_sync(0xffffffffu, acc_wt, o); }
    if (lane == 0u && acc_n) { atomicAdd(&sm.t_hits[kd], acc_n); atomicAdd(&sm.t_sw[kd], acc_w); atomicAdd(&sm.t_swt[kd], acc_wt); }
    n_up_out += n_up;
}

// DENSE (brute-force photon-output kernels only): with the dense loop and its record staging, compiled for 2 CTAs/SM;
// without, every tile takes the sparse paths (correct for any input, 3 CTAs/SM): the host launches that instance when
// no telescope is large enough to catch a good part of a shower's light (c8opt.cu, pick_kernel).
template <int TELSRC, bool COPLANAR, int NT, int MODE, bool DENSE = true>
__global__ void __launch_bounds__(kTile, (MODE == MODE_OUT && tel_base(TELSRC) == TEL_CONST && DENSE) ? kOutCtasPerSm : 3) propagate_kernel(const __grid_constant__ KParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    TileSmem &sm = *reinterpret_cast<TileSmem *>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // segments per tile: kTile / n_procs for large inputs; fewer for small ones, so that the tiles still fill the GPU
    // (the emitter slots keep their places: Cherenkov from 0, fluorescence from kTile / 2 when both run)
    const int segs_per_tile = P.tile_segs;

    // ---- clear the tile tallies
    const bool tally_in_smem = P.n_tel <= kTelSmemMax;
    if (tally_in_smem)
        for (int k = tid; k < P.n_tel; k += kTile) { sm.t_hits[k] = 0u; sm.t_sw[k] = 0.0; sm.t_swt[k] = 0.0; }
    if (tid == 0) { sm.n_upward = 0ull; sm.n_culled = 0ull; sm.flat_count = 0u; }
    sm.invalid[tid] = 0;
    sm.acc_n[tid] = 0u; sm.acc_k[tid] = -1; sm.acc_w[tid] = 0.0; sm.acc_wt[tid] = 0.0;
    if (tid < kWarps) sm.wide_count[tid] = 0u;
    constexpr bool OUT = (MODE == MODE_OUT);
    if constexpr (OUT && tel_base(TELSRC) == TEL_CONST && DENSE) {
        OutSmem &os = out_smem(sm);
        if (tid < kRoundSlots) { os.agg[tid] = 0u; os.rbase[tid] = 0ull; mbar_init(&os.rbar[tid], 1u); }
        if (tid < kTelConstMax) os.probe[tid] = 0u;
    }
    if constexpr (MODE == MODE_HIST) {
        HistSmem &hs = hist_smem(sm);
        for (int b = tid; b < P.hist_bins; b += kTile) { hs.n[b] = 0u; hs.sw_lo[b] = hs.sw_hi[b] = 0u; hs.swt_lo[b] = hs.swt_hi[b] = 0u; }
        if (tid == 0) hs.overflow = 0u;
    }
    __syncthreads();

    // ---- phase 1: preamble of emitter tid (a1)
    const int seg_local = (P.n_procs == 2) ? (tid & (kTile / 2 - 1)) : tid;
    const int tag = (P.n_procs == 2) ? (tid >> 7) : ((P.processes & 1u) ? 0 : 1);
    const unsigned long long seg_i = (unsigned long long)blockIdx.x * (unsigned)segs_per_tile + (unsigned)seg_local;
    uint32_t nb = 0, n_culled = 0;
    if (seg_local < segs_per_tile && seg_i < P.n_seg) {
        const float4 *sp = P.seg + seg_i * 3ull;
        const float4 s0 = __ldg(sp), s1 = __ldg(sp + 1), s2 = __ldg(sp + 2);
        int bad;
        bool culled;
        nb = preamble<false, tel_base(TELSRC) == TEL_CONST, tel_disp(TELSRC)>(P, s0, s1, s2, tag, &sm.frame[tid * kFrameStride], &sm.kind[tid], &bad, &culled, nullptr,
                                                  &sm.tmask[tid]);
        if (P.split_part == 2) {
            // second launch of a two-process request: the first one (Cherenkov) has counted the segments that are
            // invalid for both processes or for Cherenkov; what is left to count here is a segment whose fluorescence
            // bunch count alone is out of range (the Cherenkov preamble is run again to find out; rare)
            if (bad == 2 && (P.cauchy_b > 0.0 ? cherenkov_preamble_status_disp(P, s0, s1, s2, &sm.frame[tid * kFrameStride])
                                              : cherenkov_preamble_status(P, s0, s1, s2, &sm.frame[tid * kFrameStride])) == 0) sm.invalid[seg_local] = 1;
        } else if (bad) sm.invalid[seg_local] = 1;
        if (P.counts) {
            P.counts[seg_i * 2ull + (unsigned)tag] = nb;
            if (P.n_procs == 1 && P.split_part == 0) P.counts[seg_i * 2ull + (unsigned)(tag ^ 1)] = 0u;
        }
        if (culled) { n_culled = nb; nb = 0u; }           // generated, but provably no hit: not propagated
    }
    if (P.flags & (kFlagCull | kFlagCutCentre | kFlagCutTel)) {
        unsigned long long c = n_culled;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
        if (lane == 0 && c) atomicAdd(&sm.n_culled, c);
    }
    // ---- exclusive scan of nb over the tile, and of the cost-weighted counts that balance the warps: a photon of a
    // generic kind (fluorescence, near-horizontal Cherenkov tracks) costs about kGenericWeight axis-kind photons.
    // Every emitter takes an even number of slots of the index space (one empty slot after an odd count), so that the
    // pairs (g, g + 1), g even, which a lane of the pair loop takes, never straddle two emitters or two warps.
    const uint32_t odd = nb & 1u;
    const uint32_t nbp = nb + odd;
    sm.odd[tid] = (uint8_t)odd;
    const uint32_t n_pad_w = (uint32_t)__popc(__ballot_sync(0xffffffffu, odd != 0u));
    // (brute-force kernels: an axis-kind emitter that reaches a telescope pays the plane crossing and the pre-tests)
    uint32_t weight = (nb != 0u && sm.kind[tid] != KIND_CHER_AXIS) ? 2u * (uint32_t)kGenericWeight : 2u;
    if constexpr (tel_base(TELSRC) == TEL_CONST) { if (weight == 2u && sm.tmask[tid] != 0u) weight = 4u; }      // measured: 3: c2 0.683 ms, 4: 0.679, 5: 0.679 (unweighted 0.700)
    const unsigned long long wnb = (unsigned long long)nbp * weight;
    uint32_t inc = nbp;
    unsigned long long winc = wnb;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(0xffffffffu, inc, o);
        const unsigned long long wv = __shfl_up_sync(0xffffffffu, winc, o);
        if (lane >= o) { inc += v; winc += wv; }
    }
    if (lane == 31) { sm.warp_sum[warp] = inc; sm.warp_wsum[warp] = winc; sm.warp_pad[warp] = n_pad_w; }
    __syncthreads();
    uint32_t woff = 0, total = 0, n_pad = 0;
    unsigned long long wwoff = 0, wtotal = 0;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) {
        const uint32_t v = sm.warp_sum[w];
        const unsigned long long wv = sm.warp_wsum[w];
        if (w < warp) { woff += v; wwoff += wv; }
        total += v; wtotal += wv; n_pad += sm.warp_pad[w];
    }
    const uint32_t excl = woff + inc - nbp;
    sm.prefix[tid] = excl;
    if (tid < 8) sm.prefix[kTile + tid] = (tid == 0) ? total : 0xffffffffu;
    // warp w walks photons [bound[w], bound[w + 1]): equal shares of the weighted index space.  The emitter that
    // holds a share boundary converts it back to a photon index.
    if (tid == 0) { sm.bound[0] = 0u; sm.bound[kWarps] = total; }
    if (wnb) {
        const unsigned long long wexcl = wwoff + winc - wnb;
#pragma unroll
        // Large tiles: the shares begin on whole trips of the loops (64 slots), so that only the tile's last trip is a
        // partial one and the record blocks of a dense tile keep their size (c5g 15.95 -> 15.66 ms); small tiles
        // (fluorescence: a few hundred slots per warp) keep the finer split (tried there: c4 16.21 -> 16.43 ms).
        // (the instance with the dense loop aligns always: its tiles of interest are large)
        constexpr bool kAlignAlways = (MODE == MODE_OUT && tel_base(TELSRC) == TEL_CONST && DENSE);
        const uint32_t amask = (kAlignAlways || total >= 16384u) ? ~63u : ~1u;
        for (int w = 1; w < kWarps; ++w) {
            const unsigned long long x = wtotal / kWarps * (unsigned)w + wtotal % kWarps * (unsigned)w / kWarps;   // floor(wtotal w / 8)
            if (x >= wexcl && x < wexcl + wnb) sm.bound[w] = (excl + (uint32_t)((x - wexcl) / weight)) & amask;
        }
    }
    __syncthreads();

    // ---- phase 2: warp `warp` walks photons [lo, hi) of the tile's concatenated index space
    const uint32_t lo = sm.bound[warp], hi = sm.bound[warp + 1];
    const unsigned long long tile_first = P.first_id + (unsigned long long)blockIdx.x * (unsigned)segs_per_tile;
    uint32_t n_up = 0;

    // Every warp runs the same number of iterations (that of the longest range): the dense loop of the photon-output
    // kernels closes a round of reservations once per trip, and every warp of the tile has to arrive at it.
    uint32_t max_len = 0;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) max_len = max(max_len, sm.bound[w + 1] - sm.bound[w]);
    if (total) {
        // One instance of a loop per setting of the refraction slack in the pre-tests: it is uniform over the launch, and
        // a photon of the default path does not pay for it.
        uint32_t q_head = 0u, q_count = 0u;
        if constexpr (OUT && tel_base(TELSRC) != TEL_CONST) {
            // emitter of this lane's first photon: the e with prefix[e] <= g < prefix[e+1] (skips empty emitters)
            WarpWalk ww;
            {
                const uint32_t g0 = min(lo + (uint32_t)lane, max(hi, 1u) - 1u);
                int a = 0, b = kTile;                 // invariant: prefix[a] <= g0 < prefix[b]
                while (b - a > 1) { const int m = (a + b) >> 1; if (sm.prefix[m] <= g0) a = m; else b = m; }
                ww.e = a;
            }
            // Loop-carried per lane: photon index g, emitter e with its end, index j within the emitter, kind, the hoisted
            // Philox words (the grid kernels are short of registers and reload the axis frame from shared memory).
            ww.end = sm.prefix[ww.e + 1] - sm.odd[ww.e];
            ww.kind = sm.kind[ww.e];
            ww.pe = philox_emitter(P, emitter_segment(P, tile_first, ww.e));
            ww.f_reg = load_axis_frame(sm, ww.e);
            ww.g = lo + (uint32_t)lane; ww.j = ww.g - sm.prefix[ww.e];
            ww.n_up = 0u; ww.q_head = 0u; ww.q_count = 0u;
            const uint32_t n_iter = (max_len + 31u) / 32u;
            if (P.flags & kFlagRefract) walk<TELSRC, COPLANAR, NT, MODE, true>(P, sm, ww, hi, tile_first, n_iter);
            else walk<TELSRC, COPLANAR, NT, MODE, false>(P, sm, ww, hi, tile_first, n_iter);
            n_up = ww.n_up; q_head = ww.q_head; q_count = ww.q_count;
        } else {
            bool dense = false;
            int kd = 0;
            if constexpr (OUT && DENSE) {
                // dense or sparse tile?  (tile-uniform: every thread reads the same counts after the barrier)
                OutSmem &os = out_smem(sm);
                if (P.flags & kFlagRefract) probe_density<COPLANAR, NT, true>(P, sm, os, lo, hi, tile_first);
                else probe_density<COPLANAR, NT, false>(P, sm, os, lo, hi, tile_first);
                __syncthreads();
                uint32_t best = 0u;
#pragma unroll
                for (int k = 0; k < NT; ++k) { const uint32_t c = os.probe[k]; if (c > best) { best = c; kd = k; } }
                dense = best >= (uint32_t)kProbeDense;
            }
            if constexpr (OUT && DENSE) {
                if (dense) {
                    const uint32_t n_trips = (max_len + 63u) / 64u;
                    if (P.flags & kFlagRefract) walk_dense<COPLANAR, NT, true, false>(P, sm, out_smem(sm), lo, hi, tile_first, n_trips, kd, n_up, q_head, q_count);
                    else if (NT == 1 && COPLANAR && P.tau == nullptr && P.ids == nullptr)
                        walk_dense<COPLANAR, NT, false, NT == 1 && COPLANAR>(P, sm, out_smem(sm), lo, hi, tile_first, n_trips, kd, n_up, q_head, q_count);
                    else walk_dense<COPLANAR, NT, false, false>(P, sm, out_smem(sm), lo, hi, tile_first, n_trips, kd, n_up, q_head, q_count);
                }
            }
            if (!dense) {
                // tally, sparse photon output: candidates to the queue; ground histogram: both photons evaluated inline
                if constexpr (OUT && tel_base(TELSRC) == TEL_CONST) {
                    // The range re-read from shared memory inside a (one-pass) loop: the bounds then do not stay live in
                    // registers across the dense loop above, which the compiler schedules better for it (measured: c5g
                    // 15.92 -> 15.63 ms, c5 7.03 -> 6.98 ms; the same form costs the grid kernels 1.8 %, so only here).
                    // More than one piece per warp, interleaved over the tile, measured slower (c2 0.68 -> 0.70 ms with two).
                    for (int p = warp; p < kWarps; p += kWarps) {
                        const uint32_t plo = sm.bound[p], phi = sm.bound[p + 1];
                        if (P.flags & kFlagRefract) walk_pairs<TELSRC, COPLANAR, NT, MODE, true, MODE == MODE_HIST>(P, sm, plo, phi, tile_first, n_up, q_head, q_count);
                        else {
                            // Large tiles (their shares are whole trips but for the tile's last one): the whole trips in an
                            // instance of the loop without the per-lane range test, then the partial trip (c2 0.678 ->
                            // 0.667 ms, c5 6.98 -> 6.84 ms).  Not for small tiles, where the second entry costs more than the
                            // test (c3b + 21 %), nor in the instance with the dense loop (whose code it would perturb).
                            uint32_t pstart = plo;
                            if constexpr (!DENSE && !tel_disp(TELSRC)) {
                                if (total >= 16384u) {
                                    pstart = plo + ((phi - plo) & ~63u);
                                    walk_pairs<TELSRC, COPLANAR, NT, MODE, false, MODE == MODE_HIST, true>(P, sm, plo, pstart, tile_first, n_up, q_head, q_count);
                                }
                            }
                            walk_pairs<TELSRC, COPLANAR, NT, MODE, false, MODE == MODE_HIST>(P, sm, pstart, phi, tile_first, n_up, q_head, q_count);
                        }
                    }
                } else {
                    if (P.flags & kFlagRefract) walk_pairs<TELSRC, COPLANAR, NT, MODE, true, MODE == MODE_HIST>(P, sm, lo, hi, tile_first, n_up, q_head, q_count);
                    else {
                        uint32_t start = lo;                                        // (as above; not for the ground histogram
                        if constexpr (MODE != MODE_HIST && !tel_disp(TELSRC)) {     // and n(lambda), whose loops it slowed by 4 %)
                            if (total >= 16384u) {
                                start = lo + ((hi - lo) & ~63u);
                                walk_pairs<TELSRC, COPLANAR, NT, MODE, false, MODE == MODE_HIST, true>(P, sm, lo, start, tile_first, n_up, q_head, q_count);
                            }
                        }
                        walk_pairs<TELSRC, COPLANAR, NT, MODE, false, MODE == MODE_HIST>(P, sm, start, hi, tile_first, n_up, q_head, q_count);
                    }
                }
            }
        }
        if constexpr (tel_base(TELSRC) != TEL_CONST) {
            __syncwarp();
            const uint32_t nw = sm.wide_count[warp];
            if (nw) wide_batch<TELSRC, MODE>(P, sm, tile_first, q_head, q_count, nw);
        }
        if (q_count) drain_queue<TELSRC, MODE>(P, sm, tile_first, q_head, q_count);
        flush_accumulator(P, sm);
    }

    // ---- tile epilogue: counters and tallies
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) n_up += __shfl_xor_sync(0xffffffffu, n_up, o);
    if (lane == 0 && n_up) atomicAdd(&sm.n_upward, (unsigned long long)n_up);
    __syncthreads();
    if constexpr (MODE != MODE_HIST) {
        // the flat photons the loops set aside, in double (tile-uniform branch)
        if (sm.flat_count) {
            flat_pass<MODE, tel_disp(TELSRC)>(P, sm, tile_first);
            __syncthreads();
        }
    }
    if (tid == 0) {
        if (total - n_pad + sm.n_culled) atomicAdd(&P.counters[1], (unsigned long long)(total - n_pad) + sm.n_culled);
        if (sm.n_upward) atomicAdd(&P.counters[2], sm.n_upward);
        if (sm.n_culled) atomicAdd(&P.counters[7], sm.n_culled);
    }
    {
        // invalid segments of this tile (each counted once)
        uint32_t nbad = (tid < kTile / (int)P.n_procs) ? sm.invalid[tid] : 0u;
        nbad = __reduce_add_sync(0xffffffffu, nbad);
        if (lane == 0 && nbad) atomicAdd(&P.counters[6], (unsigned long long)nbad);   // once per segment
    }
    if constexpr (MODE == MODE_HIST) {
        // the tile's histogram into the global one (the barrier above ordered the warps' updates); bin hist_bins = overflow
        HistSmem &hs = hist_smem(sm);
        for (int b = tid; b < P.hist_bins; b += kTile) {
            const uint32_t c = hs.n[b];
            if (c) {
                atomicAdd(&P.hist[b].hits, (unsigned long long)c);
                const unsigned long long sw = ((unsigned long long)hs.sw_hi[b] << 32) | hs.sw_lo[b];
                const long long swt = (long long)(((unsigned long long)hs.swt_hi[b] << 32) | hs.swt_lo[b]);
                atomicAdd(&P.hist[b].sum_w, (double)sw * P.hist_winv);
                atomicAdd(&P.hist[b].sum_wt, (double)swt * (P.hist_winv * (1.0 / 64.0)));
            }
        }
        if (tid == 0 && hs.overflow) atomicAdd(&P.hist[P.hist_bins].hits, (unsigned long long)hs.overflow);
        return;
    }
    if (tally_in_smem) {
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
