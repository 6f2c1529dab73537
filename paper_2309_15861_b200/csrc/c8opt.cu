// c8opt.cu -- the C-ABI of include/c8opt.h: context, table upload, kernel launches.
// No torch types; device memory for segments / records is the caller's.
#include "../../include/c8opt.h"
#include "c8opt_kernels.cuh"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstddef>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

namespace {

thread_local char g_create_error[256] = "";

struct HostLayer { double h_lo, a, b, c; };

}  // namespace

struct c8opt_ctx {
    int device = 0;
    // atmosphere (host copies)
    int n_layers = 0;
    HostLayer layer[C8OPT_MAX_LAYERS];
    double eta0 = 0, rho0 = 0, h_obs = 0;
    int tau_nh = 0, tau_nl = 0;
    double tau_h0 = 0, tau_dh = 1, tau_l0 = 0, tau_dl = 1;
    float *d_tau = nullptr;
    // telescopes
    int n_tel = 0, n_tel_pending = 0;
    bool coplanar = true;
    std::vector<double> tel_xyzr;          // absolute, as given (float -> double)
    double x_ref = 0, y_ref = 0, z_ref = 0;
    double array_rb = 0;               // the same radius, exact (fluorescence beamed at the array, R28)
    int n_sm = 148;
    float cull_Rb = 0;                 // radius about the reference point that holds every telescope sphere
    // ground-plane radial profile (C8OPT_MODE_GROUND_HIST)
    c8::Tally *d_hist = nullptr;       // [hist_bins + 1], the last one counts the overflow
    int hist_bins = 0;
    double hist_core_x = 0, hist_core_y = 0, hist_r_max = 0;
    float4 *d_telA = nullptr;
    double4 *d_telD = nullptr;         // absolute centres in double (x, y, z, R): the angular particle cut (R29)
    float *d_telT = nullptr;
    float *d_telEta = nullptr;
    std::vector<float> h_telEta;
    std::vector<float4> h_telA;
    std::vector<float> h_telT;
    // ground-plane candidate grid (n_tel > kTelConstMax)
    int tel_src = c8::TEL_CONST;
    uint2 *d_grid = nullptr;
    int n_grid_levels = 0;
    c8::GridLevel grid_lvl[c8::kGridLevels + 1] = {};
    bool have_refract_grid = false;
    double refr_cmax = 0, r_max = 0;   // kappa T(lowest telescope) [m]; largest telescope radius
    // results
    // one device block, laid out for n_tel telescopes as [counters 8 x u64][cursors n x u64][tallies n x 24 B]
    // [capacity n x u64], so that a reset is one memset (all but the capacities) and a read one copy; h_results is
    // its pinned host mirror
    unsigned char *d_results = nullptr, *h_results = nullptr;
    c8::Tally *d_tallies = nullptr;
    unsigned long long *d_counters = nullptr;   // [8]
    unsigned long long *d_cursors = nullptr;    // [n_tel]
    unsigned long long *d_capacity = nullptr;   // [n_tel] capacities of the last output-mode call (device-side copy)
    bool have_capacity = false;
    unsigned long long segments_total = 0;      // host-side running count (counter 0)
    unsigned long long launches = 0;
    // host-segment pipeline
    static constexpr int kPipe = 3;             // staging buffers / internal streams of the host-segment pipeline
    cudaStream_t pipe_stream[kPipe] = {};
    cudaEvent_t pipe_event[kPipe + 1] = {};
    c8opt_segment *d_stage[kPipe] = {};
    unsigned long long stage_segments = 0;
    char error[256] = "";
};

namespace {

int fail(c8opt_ctx *ctx, int code, const char *fmt, ...)
{
    char *dst = ctx ? ctx->error : g_create_error;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 256, fmt, ap);
    va_end(ap);
    return code;
}

// Makes the context's device current for the duration of an entry point and restores the caller's device afterwards.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = (cudaSetDevice(dev) == cudaSuccess);
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
    DeviceGuard(const DeviceGuard &) = delete;
    DeviceGuard &operator=(const DeviceGuard &) = delete;
};

#define C8_CUDA(ctx, call)                                                                        \
    do {                                                                                          \
        cudaError_t e_ = (call);                                                                  \
        if (e_ != cudaSuccess)                                                                    \
            return fail(ctx, C8OPT_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e_));            \
    } while (0)

// column depth T(h) = a_i + b_i exp(-h / c_i), layer i = last one with h >= h_lo (host, fp64)
double host_depth(const c8opt_ctx *c, double h)
{
    int i = 0;
    for (int k = 1; k < c->n_layers; ++k) if (h >= c->layer[k].h_lo) i = k;
    return c->layer[i].a + c->layer[i].b * std::exp(-h / c->layer[i].c);
}

// refractivity eta(h) = eta0 rho(h) / rho0, rho = -dT/dh = (b / c) exp(-h / c) / 100 [g/cm^3] (host, fp64)
double host_refractivity(const c8opt_ctx *c, double h)
{
    int i = 0;
    for (int k = 1; k < c->n_layers; ++k) if (h >= c->layer[k].h_lo) i = k;
    return c->eta0 * (c->layer[i].b / c->layer[i].c * std::exp(-h / c->layer[i].c) / 100.0) / c->rho0;
}

// dynamic shared memory of a launch: the tile, plus the staging buffers of the brute-force photon-output kernels
// (the id staging only when the caller wants ids), or the private histogram
size_t smem_bytes(int mode, bool staging = true, bool ids = true)
{
    if (mode == c8::MODE_HIST) return sizeof(c8::TileSmem) + sizeof(c8::HistSmem);
    if (mode != c8::MODE_OUT || !staging) return sizeof(c8::TileSmem);
    (void)ids;
    return sizeof(c8::TileSmem) + sizeof(c8::OutSmem);
}

typedef void (*kernel_t)(const c8::KParams);

// out: 0 tally, 1 photon output with the dense loop, 2 photon output without it (brute-force kernels only)
template <int TELSRC, int NT> kernel_t pick_kernel2(bool coplanar, int out)
{
    if constexpr (TELSRC == c8::TEL_CONST) {
        if (out == 2)
            return coplanar ? c8::propagate_kernel<TELSRC, true, NT, c8::MODE_OUT, false> : c8::propagate_kernel<TELSRC, false, NT, c8::MODE_OUT, false>;
    }
    if (out) return coplanar ? c8::propagate_kernel<TELSRC, true, NT, c8::MODE_OUT> : c8::propagate_kernel<TELSRC, false, NT, c8::MODE_OUT>;
    return coplanar ? c8::propagate_kernel<TELSRC, true, NT, c8::MODE_TALLY> : c8::propagate_kernel<TELSRC, false, NT, c8::MODE_TALLY>;
}

// nt = number of constant-bank telescope slots the hot loop tests (n_tel rounded up to 1, 4 or 8)
int padded_count(int n_tel) { return n_tel <= 1 ? 1 : (n_tel <= 4 ? 4 : 8); }

kernel_t pick_kernel(int tel_src, bool coplanar, int nt, int out)
{
    if (tel_src == c8::TEL_CONST) {
        if (nt == 1) return pick_kernel2<c8::TEL_CONST, 1>(coplanar, out);
        if (nt == 4) return pick_kernel2<c8::TEL_CONST, 4>(coplanar, out);
        return pick_kernel2<c8::TEL_CONST, 8>(coplanar, out);
    }
    if (tel_src == c8::TEL_GRID) return pick_kernel2<c8::TEL_GRID, 0>(coplanar, out);
    return pick_kernel2<c8::TEL_GLOBAL, 0>(coplanar, out);
}

// R30 (cauchy_b_nm2 > 0): the Cherenkov launch runs on the instances with the wavelength-dependent refractive index:
// one per telescope source and mode (out: 0 tally, else photon output), the general ones -- telescopes at any height,
// eight constant-bank slots (the unused ones never hit), no dense loop.
kernel_t pick_disp_kernel(int tel_src, int out)
{
    if (tel_src == c8::TEL_CONST)
        return out ? c8::propagate_kernel<c8::TEL_CONST | c8::TEL_DISP, false, 8, c8::MODE_OUT, false>
                   : c8::propagate_kernel<c8::TEL_CONST | c8::TEL_DISP, false, 8, c8::MODE_TALLY>;
    if (tel_src == c8::TEL_GRID)
        return out ? c8::propagate_kernel<c8::TEL_GRID | c8::TEL_DISP, false, 0, c8::MODE_OUT>
                   : c8::propagate_kernel<c8::TEL_GRID | c8::TEL_DISP, false, 0, c8::MODE_TALLY>;
    return out ? c8::propagate_kernel<c8::TEL_GLOBAL | c8::TEL_DISP, false, 0, c8::MODE_OUT>
               : c8::propagate_kernel<c8::TEL_GLOBAL | c8::TEL_DISP, false, 0, c8::MODE_TALLY>;
}

// A tile of a shower's light is "dense" on a telescope (a good part of its photons hit it) only when the telescope is
// of the size of the light pool.  Below this radius the photon-output launch takes the kernel instance without the dense
// loop (3 CTAs/SM instead of 2); both instances are correct for any input.
constexpr double kDenseRadiusMin_m = 30.0;

// Ground-plane candidate grid: a photon with |v_z| >= vzmin that hits telescope k crosses the
// plane z_ref within rho_k = R / vzmin + |c_z - z_ref| sqrt(1 / vzmin^2 - 1) of (c_x, c_y).  Every cell lists the
// telescopes whose disc (plus slack for fp32 rounding) touches it; at most 4 per cell, else the resolution is
// doubled, and if that does not help this level is not built.  The cells are appended to *cells.
bool build_grid_level(c8opt_ctx *ctx, double vzmin, double extra_reach, std::vector<uint2> *cells, c8::GridLevel *lvl)
{
    const double slack = 0.05 + extra_reach;
    const int n = ctx->n_tel_pending;
    std::vector<double> rho(n);
    double x_lo = INFINITY, x_hi = -INFINITY, y_lo = INFINITY, y_hi = -INFINITY, rho_max = 0;
    for (int k = 0; k < n; ++k) {
        const double r = std::sqrt((double)ctx->h_telA[k].w), dz = std::fabs((double)ctx->h_telA[k].z);
        rho[k] = r / vzmin + dz * std::sqrt(1.0 / (vzmin * vzmin) - 1.0) + slack;
        rho_max = std::fmax(rho_max, rho[k]);
        x_lo = std::fmin(x_lo, ctx->h_telA[k].x - rho[k]); x_hi = std::fmax(x_hi, ctx->h_telA[k].x + rho[k]);
        y_lo = std::fmin(y_lo, ctx->h_telA[k].y - rho[k]); y_hi = std::fmax(y_hi, ctx->h_telA[k].y + rho[k]);
    }
    const double ext = std::fmax(x_hi - x_lo, y_hi - y_lo);
    int res = (int)std::ceil(ext / (2.0 * rho_max));
    if (res < 1) res = 1;
    if (res > 256) res = 256;
    for (; res <= 1024; res *= 2) {
        const double cell = ext / res * (1.0 + 1e-6);
        const int nx = (int)std::ceil((x_hi - x_lo) / cell), ny = (int)std::ceil((y_hi - y_lo) / cell);
        if (nx < 1 || ny < 1) return false;
        std::vector<uint16_t> list((size_t)nx * ny * 4, 0xffffu);
        bool ok = true;
        for (int k = 0; k < n && ok; ++k) {
            const double cx = ctx->h_telA[k].x - x_lo, cy = ctx->h_telA[k].y - y_lo;
            const int ix0 = std::max(0, (int)std::floor((cx - rho[k]) / cell)), ix1 = std::min(nx - 1, (int)std::floor((cx + rho[k]) / cell));
            const int iy0 = std::max(0, (int)std::floor((cy - rho[k]) / cell)), iy1 = std::min(ny - 1, (int)std::floor((cy + rho[k]) / cell));
            for (int iy = iy0; iy <= iy1 && ok; ++iy)
                for (int ix = ix0; ix <= ix1; ++ix) {
                    // distance from the disc centre to the cell rectangle (grown by 1e-3 cell against rounding of the lookup)
                    const double gx0 = (ix - 1e-3) * cell, gx1 = (ix + 1 + 1e-3) * cell, gy0 = (iy - 1e-3) * cell, gy1 = (iy + 1 + 1e-3) * cell;
                    const double ddx = std::fmax(0.0, std::fmax(gx0 - cx, cx - gx1)), ddy = std::fmax(0.0, std::fmax(gy0 - cy, cy - gy1));
                    if (ddx * ddx + ddy * ddy > rho[k] * rho[k]) continue;
                    uint16_t *c = &list[((size_t)iy * nx + ix) * 4];
                    int slot = 0;
                    while (slot < 4 && c[slot] != 0xffffu) ++slot;
                    if (slot == 4) { ok = false; break; }
                    c[slot] = (uint16_t)k;
                }
        }
        if (!ok) continue;
        const size_t base = cells->size();
        cells->resize(base + (size_t)nx * ny);
        for (size_t i = 0; i < (size_t)nx * ny; ++i)
            (*cells)[base + i] = make_uint2((uint32_t)list[4 * i] | ((uint32_t)list[4 * i + 1] << 16),
                                            (uint32_t)list[4 * i + 2] | ((uint32_t)list[4 * i + 3] << 16));
        lvl->nx = nx; lvl->ny = ny; lvl->base = (int)base;
        lvl->inv_cell = (float)(1.0 / cell); lvl->vzmin = (float)vzmin;
        lvl->ox = (float)(-x_lo * (double)lvl->inv_cell); lvl->oy = (float)(-y_lo * (double)lvl->inv_cell);
        return true;
    }
    return false;
}

// Level 0 serves |v_z| >= 0.5 (Cherenkov light of a shower), level 1 the flatter photons down to |v_z| = 0.1
// (isotropic fluorescence); what is flatter still, or has no grid, takes the kernel's wide test.
bool build_grid(c8opt_ctx *ctx, std::vector<uint2> *cells)
{
    const double vzmin[c8::kGridLevels] = {0.5, 0.1};
    ctx->n_grid_levels = 0;
    for (int l = 0; l < c8::kGridLevels; ++l) {
        if (!build_grid_level(ctx, vzmin[l], 0.0, cells, &ctx->grid_lvl[l])) break;
        ctx->n_grid_levels = l + 1;
    }
    // level 0 again for C8OPT_FLAG_REFRACT: the corrections move a photon with |v_z| >= 0.5 by up to
    // refr_cmax sin / cos^3 <= 6.93 refr_cmax in the plane (R27); if that grid cannot be built the flag is refused
    ctx->have_refract_grid = ctx->n_grid_levels > 0 &&
                             build_grid_level(ctx, vzmin[0], 7.0 * ctx->refr_cmax, cells, &ctx->grid_lvl[c8::kGridLevels]);
    return ctx->n_grid_levels > 0;
}

// Validate params / outputs and fill the kernel parameter block (everything except seg / n / first_id).
int fill_params(c8opt_ctx *ctx, const c8opt_run_params *rp, const c8opt_output *out, c8::KParams *kp)
{
    if (!rp) return fail(ctx, C8OPT_ERR_ARGUMENT, "params is NULL");
    const bool hist = rp->mode == C8OPT_MODE_GROUND_HIST;
    if (!hist && ctx->n_tel < 1) return fail(ctx, C8OPT_ERR_ARGUMENT, "no telescopes: call c8opt_add_telescopes first");
    if (hist && ctx->hist_bins < 1) return fail(ctx, C8OPT_ERR_ARGUMENT, "no histogram: call c8opt_set_ground_histogram first");
    if (hist && (rp->flags & C8OPT_FLAG_CULL)) return fail(ctx, C8OPT_ERR_ARGUMENT, "no culling in ground-histogram mode (every bunch counts)");
    if (hist && (rp->processes & C8OPT_PROC_FLUORESCENCE) && rp->fl_beam_telescope != -1)
        return fail(ctx, C8OPT_ERR_ARGUMENT, "ground-histogram mode has no telescope to beam at");
    const unsigned procs = rp->processes;
    if (procs == 0 || (procs & ~3u)) return fail(ctx, C8OPT_ERR_ARGUMENT, "processes must be a combination of bits 0 and 1");
    if (rp->mode > 2u) return fail(ctx, C8OPT_ERR_ARGUMENT, "mode must be 0 (tally), 1 (photon output) or 2 (ground histogram)");
    if (rp->flags & ~(C8OPT_FLAG_CULL | C8OPT_FLAG_REFRACT | C8OPT_FLAG_CUT_CENTRE | C8OPT_FLAG_CUT_TELESCOPES))
        return fail(ctx, C8OPT_ERR_ARGUMENT, "unknown bit in flags");
    if (rp->flags & (C8OPT_FLAG_CUT_CENTRE | C8OPT_FLAG_CUT_TELESCOPES)) {
        if (hist) return fail(ctx, C8OPT_ERR_ARGUMENT, "no particle cut in ground-histogram mode (every bunch counts)");
        if (!(rp->cut_angle_rad >= 0.0 && rp->cut_angle_rad <= 3.14159265358979323846))
            return fail(ctx, C8OPT_ERR_ARGUMENT, "cut_angle_rad must be in [0, pi]");
    }
    if (!(rp->bunch_size > 0.0) || !std::isfinite(rp->bunch_size)) return fail(ctx, C8OPT_ERR_ARGUMENT, "bunch_size must be > 0");
    if (!(rp->cauchy_b_nm2 >= 0.0) || !std::isfinite(rp->cauchy_b_nm2)) return fail(ctx, C8OPT_ERR_ARGUMENT, "cauchy_b_nm2 must be >= 0");
    if (rp->cauchy_b_nm2 > 0.0 && (procs & C8OPT_PROC_CHERENKOV)) {
        if (hist) return fail(ctx, C8OPT_ERR_ARGUMENT, "cauchy_b_nm2 > 0 is not served in ground-histogram mode");
        if (rp->flags & C8OPT_FLAG_CULL)
            return fail(ctx, C8OPT_ERR_ARGUMENT, "cauchy_b_nm2 > 0: no segment culling (the cull assumes one Cherenkov angle per segment)");
    }
    if (procs & C8OPT_PROC_CHERENKOV)
        if (!(rp->lam1_nm > 0.0) || !(rp->lam2_nm > rp->lam1_nm)) return fail(ctx, C8OPT_ERR_ARGUMENT, "need 0 < lam1 < lam2");
    if (procs & C8OPT_PROC_FLUORESCENCE) {
        if (!(rp->fl_yield_per_MeV >= 0.0) || !(rp->fl_lam1_nm > 0.0) || !(rp->fl_lam2_nm >= rp->fl_lam1_nm))
            return fail(ctx, C8OPT_ERR_ARGUMENT, "bad fluorescence yield / band");
        if (!hist && rp->fl_beam_telescope >= ctx->n_tel) return fail(ctx, C8OPT_ERR_ARGUMENT, "fl_beam_telescope out of range");
        if (rp->fl_beam_telescope >= 0 && !(rp->fl_beam_halfangle_rad > 0.0 && rp->fl_beam_halfangle_rad <= 3.14159265358979323846))
            return fail(ctx, C8OPT_ERR_ARGUMENT, "fl_beam_halfangle_rad must be in (0, pi]");
    }
    if (rp->mode == C8OPT_MODE_OUTPUT && (!out || !out->records || !out->tel_offset || !out->tel_capacity))
        return fail(ctx, C8OPT_ERR_ARGUMENT, "photon-output mode needs out->records, tel_offset and tel_capacity");

    c8::KParams &P = *kp;
    std::memset(&P, 0, sizeof(P));
    P.n_layers = ctx->n_layers;
    for (int i = 0; i < ctx->n_layers; ++i) {
        P.layer[i] = c8::LayerD{ctx->layer[i].h_lo, ctx->layer[i].a, ctx->layer[i].b, ctx->layer[i].c};
        P.layerf[i] = c8::LayerF{(float)ctx->layer[i].h_lo, (float)ctx->layer[i].a, (float)ctx->layer[i].b,
                                 (float)(1.4426950408889634 / ctx->layer[i].c)};
    }
    P.eta0 = ctx->eta0; P.rho0 = ctx->rho0;
    P.kappa_m = (float)(0.01 * ctx->eta0 / ctx->rho0);
    P.tau = ctx->d_tau; P.tau_nh = ctx->tau_nh; P.tau_nl = ctx->tau_nl;
    P.tau_h0 = (float)ctx->tau_h0; P.tau_inv_dh = (float)(1.0 / ctx->tau_dh);
    P.tau_l0 = (float)ctx->tau_l0; P.tau_inv_dl = (float)(1.0 / ctx->tau_dl);
    P.tau_h0_d = ctx->tau_h0; P.tau_dh_d = ctx->tau_dh; P.tau_l0_d = ctx->tau_l0; P.tau_dl_d = ctx->tau_dl;
    P.lam1_d = rp->lam1_nm; P.lam2_d = rp->lam2_nm; P.fl_lam1_d = rp->fl_lam1_nm; P.fl_lam2_d = rp->fl_lam2_nm;
    P.n_tel = ctx->n_tel; P.telA = ctx->d_telA; P.telT = ctx->d_telT; P.telEta = ctx->d_telEta;
    if (ctx->tel_src == c8::TEL_CONST) {
        for (int k = 0; k < c8::kTelConstMax; ++k) { P.tel_c[k] = make_float4(0.f, 0.f, 0.f, -1.f); P.telT_c[k] = 0.f; }   // R^2 = -1: never hit
        for (int k = 0; k < ctx->n_tel; ++k) { P.tel_c[k] = ctx->h_telA[k]; P.telT_c[k] = ctx->h_telT[k]; P.telEta_c[k] = ctx->h_telEta[k]; }
    }
    P.grid = ctx->d_grid; P.n_grid_levels = ctx->n_grid_levels;
    for (int l = 0; l <= c8::kGridLevels; ++l) P.grid_lvl[l] = ctx->grid_lvl[l];
    P.x_ref = ctx->x_ref; P.y_ref = ctx->y_ref; P.z_ref = ctx->z_ref; P.z_ref_f = (float)ctx->z_ref;
    for (int i = ctx->n_layers; i < c8::kMaxLayers; ++i) P.layerf[i].h_lo = INFINITY;   // never selected by the layer count
    for (int r = 0; r < 10; ++r) {
        P.rk0[r] = (uint32_t)rp->seed + (uint32_t)r * 0x9E3779B9u;
        P.rk1[r] = (uint32_t)(rp->seed >> 32) + (uint32_t)r * 0xBB67AE85u;
    }
    P.processes = procs; P.n_procs = (procs == 3u) ? 2u : 1u;
    P.flags = rp->flags; P.cull_Rb = ctx->cull_Rb;
    P.telD = ctx->d_telD;
    P.cut_cos = (rp->flags & (C8OPT_FLAG_CUT_CENTRE | C8OPT_FLAG_CUT_TELESCOPES)) ? std::cos(rp->cut_angle_rad) : -2.0;
    if (rp->flags & C8OPT_FLAG_REFRACT) {
        if (ctx->tel_src == c8::TEL_GRID && !ctx->have_refract_grid && !hist)
            return fail(ctx, C8OPT_ERR_ARGUMENT, "C8OPT_FLAG_REFRACT: no candidate grid with the refraction reach can be built for this array");
        P.refr_cmax = (float)ctx->refr_cmax; P.refr_two_rmax = (float)(2.0 * ctx->r_max);
    }
    if (procs & C8OPT_PROC_CHERENKOV) {
        // PAPER.md:45 prefactor: pi e^2 / (h eps0 c0) = 2 pi alpha; the lambda integral of lambda^-2 in closed form (R2)
        const double two_pi_alpha = 2.0 * 3.14159265358979323846 * 7.2973525693e-3;
        P.c_ft = two_pi_alpha * (1.0 / rp->lam1_nm - 1.0 / rp->lam2_nm) * 1.0e9;
        P.inv_lam1 = (float)(1.0 / rp->lam1_nm);
        P.dinv_lam = (float)(1.0 / rp->lam1_nm - 1.0 / rp->lam2_nm);
        // R30: n(lambda, h) - 1 = eta(h) (1 + b / lambda^2); the yield integral runs over x = 1 / lambda in the preamble
        P.cauchy_b = rp->cauchy_b_nm2; P.cauchy_b_f = (float)rp->cauchy_b_nm2;
        P.x1_d = 1.0 / rp->lam1_nm; P.x2_d = 1.0 / rp->lam2_nm;
        P.c_ft0 = two_pi_alpha * 1.0e9;
    }
    P.bunch_size = rp->bunch_size; P.fl_yield = rp->fl_yield_per_MeV;
    P.fl_lam1 = (float)rp->fl_lam1_nm; P.fl_dlam = (float)(rp->fl_lam2_nm - rp->fl_lam1_nm);
    P.beam_tel = (procs & C8OPT_PROC_FLUORESCENCE) ? rp->fl_beam_telescope : -1;
    if (P.beam_tel < -2) return fail(ctx, C8OPT_ERR_ARGUMENT, "fl_beam_telescope must be >= -2");
    if (P.beam_tel == C8OPT_BEAM_ARRAY) {
        P.beam_x = ctx->x_ref; P.beam_y = ctx->y_ref; P.beam_z = ctx->z_ref; P.beam_rb = ctx->array_rb;
    }
    if (P.beam_tel >= 0) {
        P.beam_x = ctx->tel_xyzr[4 * P.beam_tel + 0]; P.beam_y = ctx->tel_xyzr[4 * P.beam_tel + 1];
        P.beam_z = ctx->tel_xyzr[4 * P.beam_tel + 2];
        const double sh = std::sin(0.5 * rp->fl_beam_halfangle_rad);
        P.omc = 2.0 * sh * sh;
    }
    P.tallies = ctx->d_tallies; P.counters = ctx->d_counters; P.cursors = ctx->d_cursors;
    if (hist) {
        // R26: the profile is taken on the observation level about the core; the kernel sees one accept-all detector
        // there (R^2 = 1e30), so a hit's (x, y) is the plane crossing relative to the core.
        P.n_tel = 1; P.telA = nullptr; P.telT = nullptr; P.tallies = nullptr; P.cursors = nullptr;
        for (int k = 0; k < c8::kTelConstMax; ++k) { P.tel_c[k] = make_float4(0.f, 0.f, 0.f, -1.f); P.telT_c[k] = 0.f; }
        P.tel_c[0] = make_float4(0.f, 0.f, 0.f, 1e30f);
        P.telT_c[0] = (float)host_depth(ctx, ctx->h_obs);
        P.telEta_c[0] = (float)host_refractivity(ctx, ctx->h_obs); P.telEta = nullptr;
        P.x_ref = ctx->hist_core_x; P.y_ref = ctx->hist_core_y; P.z_ref = ctx->h_obs; P.z_ref_f = (float)ctx->h_obs;
        P.n_grid_levels = 0; P.grid = nullptr;
        if (rp->flags & C8OPT_FLAG_REFRACT) P.refr_cmax = (float)(0.01 * ctx->eta0 / ctx->rho0 * host_depth(ctx, ctx->h_obs));
        P.hist = ctx->d_hist; P.hist_bins = ctx->hist_bins; P.hist_inv_dr = (float)(ctx->hist_bins / ctx->hist_r_max);
        P.hist_wscale = (float)(65536.0 / rp->bunch_size); P.hist_winv = 1.0 / (double)P.hist_wscale;
    }
    if (out) {
        if (rp->mode == C8OPT_MODE_OUTPUT) {
            P.records = out->records; P.tel_offset = (const unsigned long long *)out->tel_offset;
            P.tel_capacity = (const unsigned long long *)out->tel_capacity; P.ids = (unsigned long long *)out->ids;
        }
        P.counts = out->counts;
    }
    return C8OPT_OK;
}

int launch_one(c8opt_ctx *ctx, c8::KParams &P, unsigned mode, unsigned long long n, cudaStream_t st)
{
    // Full tiles for large inputs; small inputs are cut into about one wave of tiles (3 CTAs on each of the SMs), at
    // least 8 segments each, so that 10^4 segments do not run on a quarter of the GPU.
    // At most kTile - 1 segments per tile: the tile's photon index space is 32 bits wide and an emitter holds up to
    // 2^24 - 1 bunches (R23), padded to 2^24 slots, so 255 emitters stay below 2^32 - 2^24 whatever their counts.
    const unsigned long long per_tile_max = (c8::kTile - 1) / P.n_procs;
    const unsigned long long one_wave = 3ull * (unsigned long long)ctx->n_sm;
    unsigned long long per_tile = (n + one_wave - 1) / one_wave;
    per_tile = std::min(per_tile_max, std::max(8ull, per_tile));
    P.tile_segs = (int)per_tile;
    const unsigned long long tiles = (n + per_tile - 1) / per_tile;
    if (tiles > 0x7fffffffull) return fail(ctx, C8OPT_ERR_ARGUMENT, "too many segments in one call");
    if (mode == C8OPT_MODE_GROUND_HIST) {
        // one accept-all detector on the observation level: brute-force kernel with a single coplanar slot
        c8::propagate_kernel<c8::TEL_CONST, true, 1, c8::MODE_HIST><<<(unsigned)tiles, c8::kTile, smem_bytes(c8::MODE_HIST), st>>>(P);
    } else {
        const bool out = P.records != nullptr;
        const bool dense_loop = out && ctx->tel_src == c8::TEL_CONST && ctx->r_max >= kDenseRadiusMin_m;
        const bool disp = P.cauchy_b > 0.0 && (P.processes & C8OPT_PROC_CHERENKOV);
        if (disp) {
            pick_disp_kernel(ctx->tel_src, out)<<<(unsigned)tiles, c8::kTile, smem_bytes(out ? c8::MODE_OUT : c8::MODE_TALLY, false), st>>>(P);
        } else {
            kernel_t k = pick_kernel(ctx->tel_src, ctx->coplanar, padded_count(ctx->n_tel), out ? (dense_loop || ctx->tel_src != c8::TEL_CONST ? 1 : 2) : 0);
            k<<<(unsigned)tiles, c8::kTile, smem_bytes(out ? c8::MODE_OUT : c8::MODE_TALLY, dense_loop, P.ids != nullptr), st>>>(P);
        }
    }
    C8_CUDA(ctx, cudaGetLastError());
    ctx->launches += 1;
    return C8OPT_OK;
}

int launch(c8opt_ctx *ctx, c8::KParams &P, unsigned mode, const c8opt_segment *d_seg, unsigned long long n,
           unsigned long long first_id, uint32_t *counts, cudaStream_t st)
{
    if (n == 0) return C8OPT_OK;
    P.seg = reinterpret_cast<const float4 *>(d_seg);
    P.n_seg = n; P.first_id = first_id; P.counts = counts;
    int rc;
    if (P.n_procs == 2) {
        // Both processes: one launch per process on the same stream (Cherenkov, then fluorescence).  The photons are
        // the same (the random stream is keyed by the process tag), but tiles of one kind only are balanced without
        // the cost weights and the Cherenkov tiles hold twice the segments: c4 17.9 -> 16.8 ms.
        c8::KParams Q = P;
        Q.n_procs = 1; Q.processes = C8OPT_PROC_CHERENKOV; Q.split_part = 1;
        rc = launch_one(ctx, Q, mode, n, st);
        if (rc != C8OPT_OK) return rc;
        Q.processes = C8OPT_PROC_FLUORESCENCE; Q.split_part = 2;
        rc = launch_one(ctx, Q, mode, n, st);
    } else {
        P.split_part = 0;
        rc = launch_one(ctx, P, mode, n, st);
    }
    if (rc != C8OPT_OK) return rc;
    ctx->segments_total += n;
    return C8OPT_OK;
}

// Photon-output mode: keep the capacities of this call for c8opt_read_tallies (records kept / dropped per telescope).
// Device-to-device into the context's own buffer, asynchronous on the caller's stream: no host synchronisation on
// the hot call, and the caller's tel_capacity array need not outlive it.
int remember_capacity(c8opt_ctx *ctx, const c8opt_run_params *rp, const c8opt_output *out, cudaStream_t st)
{
    if (rp->mode != C8OPT_MODE_OUTPUT) return C8OPT_OK;
    C8_CUDA(ctx, cudaMemcpyAsync(ctx->d_capacity, out->tel_capacity, sizeof(unsigned long long) * ctx->n_tel,
                                 cudaMemcpyDeviceToDevice, st));
    ctx->have_capacity = true;
    return C8OPT_OK;
}

// The internal streams, their events and the device staging buffers of c8opt_propagate_segments_host.
int ensure_pipeline(c8opt_ctx *ctx, unsigned long long chunk_segments)
{
    if (!ctx->pipe_stream[0]) {
        for (int i = 0; i < c8opt_ctx::kPipe; ++i) C8_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->pipe_stream[i], cudaStreamNonBlocking));
        for (int i = 0; i <= c8opt_ctx::kPipe; ++i) C8_CUDA(ctx, cudaEventCreateWithFlags(&ctx->pipe_event[i], cudaEventDisableTiming));
    }
    if (ctx->stage_segments < chunk_segments) {
        for (int i = 0; i < c8opt_ctx::kPipe; ++i) {
            C8_CUDA(ctx, cudaStreamSynchronize(ctx->pipe_stream[i]));
            cudaFree(ctx->d_stage[i]); ctx->d_stage[i] = nullptr;
        }
        ctx->stage_segments = 0;
        for (int i = 0; i < c8opt_ctx::kPipe; ++i) C8_CUDA(ctx, cudaMalloc(&ctx->d_stage[i], sizeof(c8opt_segment) * chunk_segments));
        ctx->stage_segments = chunk_segments;
    }
    return C8OPT_OK;
}

// largest chunk of the host-segment pipeline: a quarter of the table, between 32 Ki and 1 Mi segments, whole tiles
unsigned long long host_chunk_max(unsigned long long n)
{
    unsigned long long chunk = (n + 3) / 4;
    if (chunk < (1ull << 15)) chunk = 1ull << 15;
    if (chunk > (1ull << 20)) chunk = 1ull << 20;
    return (chunk + c8::kTile - 1) / c8::kTile * c8::kTile;
}

}  // namespace

extern "C" {

int c8opt_create_atmosphere(const c8opt_atmosphere_desc *desc, c8opt_ctx **out)
{
    if (!desc || !out) return fail(nullptr, C8OPT_ERR_ARGUMENT, "desc or out is NULL");
    *out = nullptr;
    if (desc->n_layers < 1 || desc->n_layers > C8OPT_MAX_LAYERS) return fail(nullptr, C8OPT_ERR_ARGUMENT, "n_layers out of range");
    for (int i = 0; i < desc->n_layers; ++i) {
        const c8opt_layer &l = desc->layers[i];
        if (!std::isfinite(l.h_lo_m) || !std::isfinite(l.a_gcm2) || !std::isfinite(l.b_gcm2) || !(l.c_m > 0.0) || !std::isfinite(l.c_m))
            return fail(nullptr, C8OPT_ERR_ARGUMENT, "layer %d: non-finite coefficient or c <= 0", i);
        if (i > 0 && !(l.h_lo_m > desc->layers[i - 1].h_lo_m)) return fail(nullptr, C8OPT_ERR_ARGUMENT, "layer bounds must ascend");
    }
    if (!(desc->rho0_gcm3 > 0.0) || !std::isfinite(desc->eta0) || !(desc->eta0 >= 0.0) || !std::isfinite(desc->h_obs_m))
        return fail(nullptr, C8OPT_ERR_ARGUMENT, "need rho0 > 0, eta0 >= 0, finite h_obs");
    const bool has_tau = desc->tau != nullptr && desc->tau_nh > 0;
    if (has_tau) {
        if (desc->tau_nl < 1 || desc->tau_nh > 4096 || desc->tau_nl > 4096 || !(desc->tau_dh_m > 0.0) || !(desc->tau_dl_nm > 0.0))
            return fail(nullptr, C8OPT_ERR_ARGUMENT, "bad transmission table shape / spacing");
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(nullptr, C8OPT_ERR_CUDA, "no CUDA device (this library has no CPU fallback)");
    }
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess)
        return fail(nullptr, C8OPT_ERR_CUDA, "cannot query the current CUDA device");
    if (prop.major != 10) return fail(nullptr, C8OPT_ERR_CUDA, "device is sm_%d%d, this library is built for sm_100a only", prop.major, prop.minor);

    c8opt_ctx *ctx = new (std::nothrow) c8opt_ctx();
    if (!ctx) return fail(nullptr, C8OPT_ERR_ARGUMENT, "out of host memory");
    ctx->device = dev;
    ctx->n_sm = prop.multiProcessorCount > 0 ? prop.multiProcessorCount : 148;
    ctx->n_layers = desc->n_layers;
    for (int i = 0; i < desc->n_layers; ++i)
        ctx->layer[i] = HostLayer{desc->layers[i].h_lo_m, desc->layers[i].a_gcm2, desc->layers[i].b_gcm2, desc->layers[i].c_m};
    ctx->eta0 = desc->eta0; ctx->rho0 = desc->rho0_gcm3; ctx->h_obs = desc->h_obs_m;
    cudaError_t e = cudaSuccess;
    if (has_tau) {
        ctx->tau_nh = desc->tau_nh; ctx->tau_nl = desc->tau_nl;
        ctx->tau_h0 = desc->tau_h0_m; ctx->tau_dh = desc->tau_dh_m; ctx->tau_l0 = desc->tau_l0_nm; ctx->tau_dl = desc->tau_dl_nm;
        const size_t bytes = sizeof(float) * (size_t)desc->tau_nh * (size_t)desc->tau_nl;
        e = cudaMalloc(&ctx->d_tau, bytes);
        if (e == cudaSuccess) e = cudaMemcpy(ctx->d_tau, desc->tau, bytes, cudaMemcpyHostToDevice);
    }
    const size_t results_bytes = 64 + (size_t)C8OPT_MAX_TELESCOPES * (8 + sizeof(c8::Tally) + 8);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_results, results_bytes);
    if (e == cudaSuccess) e = cudaMemset(ctx->d_results, 0, results_bytes);
    if (e == cudaSuccess) e = cudaMallocHost(&ctx->h_results, results_bytes);
    ctx->d_counters = reinterpret_cast<unsigned long long *>(ctx->d_results);
    for (int ts = 0; ts < 3 && e == cudaSuccess; ++ts)
        for (int nt = 1; nt <= 8 && e == cudaSuccess; nt *= (nt == 1 ? 4 : 2))
            for (int cp = 0; cp < 4 && e == cudaSuccess; ++cp)
                e = cudaFuncSetAttribute(pick_kernel(ts, (cp & 1) != 0, nt, (cp & 2) ? 1 : 0), cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem_bytes((cp & 2) ? c8::MODE_OUT : c8::MODE_TALLY));
    for (int nt = 1; nt <= 8 && e == cudaSuccess; nt *= (nt == 1 ? 4 : 2))
        for (int cp = 0; cp < 2 && e == cudaSuccess; ++cp)
            e = cudaFuncSetAttribute(pick_kernel(c8::TEL_CONST, cp != 0, nt, 2), cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     (int)smem_bytes(c8::MODE_OUT, false));
    for (int ts = 0; ts < 3 && e == cudaSuccess; ++ts)
        for (int o = 0; o < 2 && e == cudaSuccess; ++o)
            e = cudaFuncSetAttribute(pick_disp_kernel(ts, o), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes(o ? c8::MODE_OUT : c8::MODE_TALLY, false));
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(c8::propagate_kernel<c8::TEL_CONST, true, 1, c8::MODE_HIST>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)smem_bytes(c8::MODE_HIST));
    if (e != cudaSuccess) {
        fail(nullptr, C8OPT_ERR_CUDA, "context setup: %s", cudaGetErrorString(e));
        c8opt_destroy(ctx);
        return C8OPT_ERR_CUDA;
    }
    *out = ctx;
    return C8OPT_OK;
}

int c8opt_add_telescopes(c8opt_ctx *ctx, const float *xyzr, int32_t n)
{
    if (!ctx) return C8OPT_ERR_ARGUMENT;
    if (!xyzr) return fail(ctx, C8OPT_ERR_ARGUMENT, "xyzr is NULL");
    if (n < 1 || n > C8OPT_MAX_TELESCOPES) return fail(ctx, C8OPT_ERR_ARGUMENT, "telescope count %d out of range 1..%d", n, C8OPT_MAX_TELESCOPES);
    double lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    for (int k = 0; k < n; ++k) {
        for (int i = 0; i < 4; ++i)
            if (!std::isfinite(xyzr[4 * k + i])) return fail(ctx, C8OPT_ERR_ARGUMENT, "telescope %d: non-finite value", k);
        if (!(xyzr[4 * k + 3] > 0.0f)) return fail(ctx, C8OPT_ERR_ARGUMENT, "telescope %d: radius must be > 0", k);
        for (int i = 0; i < 3; ++i) { lo[i] = std::fmin(lo[i], xyzr[4 * k + i]); hi[i] = std::fmax(hi[i], xyzr[4 * k + i]); }
    }
    DeviceGuard guard(ctx->device);
    C8_CUDA(ctx, cudaDeviceSynchronize());
    ctx->n_tel = 0;
    cudaFree(ctx->d_telA); cudaFree(ctx->d_telT); cudaFree(ctx->d_telEta); cudaFree(ctx->d_grid); cudaFree(ctx->d_telD);
    ctx->d_telA = nullptr; ctx->d_telT = nullptr; ctx->d_telEta = nullptr; ctx->d_grid = nullptr; ctx->d_telD = nullptr;
    ctx->tel_xyzr.assign(xyzr, xyzr + 4 * (size_t)n);
    // reference point: centre of the bounding box; all device coordinates are relative to it
    ctx->x_ref = 0.5 * (lo[0] + hi[0]); ctx->y_ref = 0.5 * (lo[1] + hi[1]); ctx->z_ref = 0.5 * (lo[2] + hi[2]);
    ctx->coplanar = (lo[2] == hi[2]);
    std::vector<float4> &A = ctx->h_telA;
    std::vector<float> &T = ctx->h_telT;
    A.resize(n); T.resize(n);
    for (int k = 0; k < n; ++k) {
        const double x = xyzr[4 * k], y = xyzr[4 * k + 1], z = xyzr[4 * k + 2], r = xyzr[4 * k + 3];
        A[k] = make_float4((float)(x - ctx->x_ref), (float)(y - ctx->y_ref), (float)(z - ctx->z_ref), (float)(r * r));
        T[k] = (float)host_depth(ctx, z);
    }
    {
        double z_low = INFINITY;
        ctx->r_max = 0.0;
        for (int k = 0; k < n; ++k) { z_low = std::fmin(z_low, xyzr[4 * k + 2]); ctx->r_max = std::fmax(ctx->r_max, xyzr[4 * k + 3]); }
        ctx->refr_cmax = 0.01 * ctx->eta0 / ctx->rho0 * host_depth(ctx, z_low);
    }
    ctx->h_telEta.resize(n);
    for (int k = 0; k < n; ++k) ctx->h_telEta[k] = (float)host_refractivity(ctx, xyzr[4 * k + 2]);
    double rb = 0.0;
    for (int k = 0; k < n; ++k) {
        const double x = xyzr[4 * k] - ctx->x_ref, y = xyzr[4 * k + 1] - ctx->y_ref, z = xyzr[4 * k + 2] - ctx->z_ref;
        rb = std::fmax(rb, std::sqrt(x * x + y * y + z * z) + xyzr[4 * k + 3]);
    }
    ctx->cull_Rb = (float)(rb * (1.0 + 1e-6));
    ctx->array_rb = rb;
    C8_CUDA(ctx, cudaMalloc(&ctx->d_telA, sizeof(float4) * n));
    C8_CUDA(ctx, cudaMalloc(&ctx->d_telT, sizeof(float) * n));
    C8_CUDA(ctx, cudaMalloc(&ctx->d_telEta, sizeof(float) * n));
    ctx->d_cursors = reinterpret_cast<unsigned long long *>(ctx->d_results + 64);
    ctx->d_tallies = reinterpret_cast<c8::Tally *>(ctx->d_results + 64 + 8 * (size_t)n);
    ctx->d_capacity = reinterpret_cast<unsigned long long *>(ctx->d_results + 64 + 32 * (size_t)n);
    {
        std::vector<double4> D(n);
        for (int k = 0; k < n; ++k) D[k] = make_double4(xyzr[4 * k], xyzr[4 * k + 1], xyzr[4 * k + 2], xyzr[4 * k + 3]);
        C8_CUDA(ctx, cudaMalloc(&ctx->d_telD, sizeof(double4) * n));
        C8_CUDA(ctx, cudaMemcpy(ctx->d_telD, D.data(), sizeof(double4) * n, cudaMemcpyHostToDevice));
    }
    C8_CUDA(ctx, cudaMemcpy(ctx->d_telA, A.data(), sizeof(float4) * n, cudaMemcpyHostToDevice));
    C8_CUDA(ctx, cudaMemcpy(ctx->d_telT, T.data(), sizeof(float) * n, cudaMemcpyHostToDevice));
    C8_CUDA(ctx, cudaMemcpy(ctx->d_telEta, ctx->h_telEta.data(), sizeof(float) * n, cudaMemcpyHostToDevice));
    ctx->tel_src = c8::TEL_CONST;
    if (n >= c8::kTelGridMin) {
        // the grid lookup costs more than four brute-force pre-tests (11 instructions each), so it serves from
        // kTelGridMin = 9 telescopes up (tried at 3: c2 1.07 -> 1.26 ms)
        std::vector<uint2> cells;
        ctx->n_tel_pending = n;
        if (build_grid(ctx, &cells)) {
            C8_CUDA(ctx, cudaMalloc(&ctx->d_grid, sizeof(uint2) * cells.size()));
            C8_CUDA(ctx, cudaMemcpy(ctx->d_grid, cells.data(), sizeof(uint2) * cells.size(), cudaMemcpyHostToDevice));
            ctx->tel_src = c8::TEL_GRID;
        } else if (n > c8::kTelConstMax) {
            ctx->tel_src = c8::TEL_GLOBAL;
        }
    }
    ctx->n_tel = n;
    ctx->have_capacity = false;
    const int rc = c8opt_reset_tallies(ctx, nullptr);
    if (rc != C8OPT_OK) return rc;
    C8_CUDA(ctx, cudaDeviceSynchronize());
    return C8OPT_OK;
}

int c8opt_propagate_segments(c8opt_ctx *ctx, const c8opt_segment *d_seg, uint64_t n, uint64_t first_segment_id,
                             const c8opt_run_params *params, const c8opt_output *out, void *cuda_stream)
{
    if (!ctx) return C8OPT_ERR_ARGUMENT;
    if (!d_seg && n) return fail(ctx, C8OPT_ERR_ARGUMENT, "d_seg is NULL");
    DeviceGuard guard(ctx->device);
    c8::KParams P;
    int rc = fill_params(ctx, params, out, &P);
    if (rc != C8OPT_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    rc = remember_capacity(ctx, params, out, st);
    if (rc != C8OPT_OK) return rc;
    return launch(ctx, P, params->mode, d_seg, n, first_segment_id, out ? out->counts : nullptr, st);
}

int c8opt_reserve_host_staging(c8opt_ctx *ctx, uint64_t max_segments)
{
    if (!ctx) return C8OPT_ERR_ARGUMENT;
    DeviceGuard guard(ctx->device);
    return ensure_pipeline(ctx, host_chunk_max(max_segments));
}

int c8opt_propagate_segments_host(c8opt_ctx *ctx, const c8opt_segment *h_seg, uint64_t n, uint64_t first_segment_id,
                                  const c8opt_run_params *params, const c8opt_output *out, void *cuda_stream)
{
    if (!ctx) return C8OPT_ERR_ARGUMENT;
    if (!h_seg && n) return fail(ctx, C8OPT_ERR_ARGUMENT, "h_seg is NULL");
    DeviceGuard guard(ctx->device);
    c8::KParams P;
    int rc = fill_params(ctx, params, out, &P);
    if (rc != C8OPT_OK) return rc;
    cudaStream_t user = (cudaStream_t)cuda_stream;
    rc = remember_capacity(ctx, params, out, user);
    if (rc != C8OPT_OK) return rc;
    if (n == 0) return C8OPT_OK;
    // Chunk schedule: the first chunk is small (1/12 of the table, between 32 Ki and 256 Ki segments; measured on c2, 10^6
    // segments, end to end: 1/32: 1.058 ms, 1/16: 1.035, 1/12: 1.026, 1/8: 1.063) so that the first kernel
    // starts after a short copy; the chunks then double up to a quarter of the table, so that the kernels in the
    // middle fill the GPU for several waves, and no chunk takes more than a quarter of what is left, so that the last
    // kernels, which no copy overlaps, are short again (a half: 1.085 ms end to end on c2, a third: 1.063, a quarter:
    // 1.050; the copy alone takes 0.88 ms, in these chunks 0.92).  Three staging buffers, copy and kernel of a chunk on
    // the same internal stream: the copy of chunk c + 3 waits for the kernel of chunk c (with two buffers the copy
    // engine stood still in the tapering part, where the kernel of a chunk outlasts the copy of the next: 1.158 ms).
    const unsigned long long chunk_max = host_chunk_max(n);
    rc = ensure_pipeline(ctx, chunk_max);          // allocates on the first call unless c8opt_reserve_host_staging did
    if (rc != C8OPT_OK) return rc;
    unsigned long long chunk_min = (n + 11) / 12;
    if (chunk_min < (1ull << 15)) chunk_min = 1ull << 15;
    if (chunk_min > (1ull << 18)) chunk_min = 1ull << 18;
    chunk_min = (chunk_min + c8::kTile - 1) / c8::kTile * c8::kTile;
    if (chunk_min > chunk_max) chunk_min = chunk_max;
    unsigned long long grow = chunk_min;
    constexpr int kPipe = c8opt_ctx::kPipe;
    C8_CUDA(ctx, cudaEventRecord(ctx->pipe_event[kPipe], user));
    for (int i = 0; i < kPipe; ++i) C8_CUDA(ctx, cudaStreamWaitEvent(ctx->pipe_stream[i], ctx->pipe_event[kPipe], 0));
    int c = 0;
    cudaError_t ce = cudaSuccess;
    for (unsigned long long off = 0, m = 0; off < n && rc == C8OPT_OK && ce == cudaSuccess; off += m, grow = std::min(2 * grow, chunk_max), ++c) {
        const unsigned long long left = n - off, half = (left / 4 + c8::kTile - 1) / c8::kTile * c8::kTile;   // (a quarter)
        m = std::min(left, std::max(chunk_min, std::min(grow, half)));
        cudaStream_t st = ctx->pipe_stream[c % kPipe];
        ce = cudaMemcpyAsync(ctx->d_stage[c % kPipe], h_seg + off, sizeof(c8opt_segment) * m, cudaMemcpyHostToDevice, st);
        if (ce != cudaSuccess) break;
        rc = launch(ctx, P, params->mode, ctx->d_stage[c % kPipe], m, first_segment_id + off,
                    (out && out->counts) ? out->counts + 2 * off : nullptr, st);
    }
    // also after an error: the caller's stream waits for whatever was enqueued on the internal streams
    for (int i = 0; i < kPipe; ++i) {
        const cudaError_t e1 = cudaEventRecord(ctx->pipe_event[i], ctx->pipe_stream[i]);
        const cudaError_t e2 = (e1 == cudaSuccess) ? cudaStreamWaitEvent(user, ctx->pipe_event[i], 0) : e1;
        if (ce == cudaSuccess && e2 != cudaSuccess) ce = e2;
    }
    if (rc != C8OPT_OK) return rc;
    if (ce != cudaSuccess) return fail(ctx, C8OPT_ERR_CUDA, "host-segment pipeline: %s", cudaGetErrorString(ce));
    return C8OPT_OK;
}

int c8opt_read_tallies(c8opt_ctx *ctx, c8opt_tally *host_out, int32_t n_tel, uint64_t *counters, uint64_t *host_tel_count)
{
    if (!ctx) return C8OPT_ERR_ARGUMENT;
    if (!host_out) return fail(ctx, C8OPT_ERR_ARGUMENT, "host_out is NULL");
    if (n_tel != ctx->n_tel || n_tel < 1) return fail(ctx, C8OPT_ERR_ARGUMENT, "n_tel = %d but the context has %d telescopes", n_tel, ctx->n_tel);
    DeviceGuard guard(ctx->device);
    C8_CUDA(ctx, cudaDeviceSynchronize());
    static_assert(sizeof(c8opt_tally) == sizeof(c8::Tally), "tally layout");
    // one copy of the whole result block into its pinned mirror
    C8_CUDA(ctx, cudaMemcpy(ctx->h_results, ctx->d_results, 64 + 40 * (size_t)n_tel, cudaMemcpyDeviceToHost));
    const unsigned long long *cnt = reinterpret_cast<const unsigned long long *>(ctx->h_results);
    const unsigned long long *cur = cnt + 8;
    std::memcpy(host_out, ctx->h_results + 64 + 8 * (size_t)n_tel, sizeof(c8::Tally) * n_tel);
    std::vector<unsigned long long> capacity(n_tel, ~0ull);
    if (ctx->have_capacity) std::memcpy(capacity.data(), ctx->h_results + 64 + 32 * (size_t)n_tel, 8 * (size_t)n_tel);
    unsigned long long hits = 0, stored = 0, dropped = 0;
    for (int k = 0; k < n_tel; ++k) {
        hits += host_out[k].hits;
        unsigned long long kept = cur[k];
        if (kept > capacity[k]) { dropped += kept - capacity[k]; kept = capacity[k]; }
        stored += kept;
        if (host_tel_count) host_tel_count[k] = kept;
    }
    if (counters) {
        counters[C8OPT_CNT_SEGMENTS] = ctx->segments_total;
        counters[C8OPT_CNT_GENERATED] = cnt[1];
        counters[C8OPT_CNT_UPWARD] = cnt[2];
        counters[C8OPT_CNT_HITS] = hits;
        counters[C8OPT_CNT_RECORDS] = stored;
        counters[C8OPT_CNT_DROPPED] = dropped;
        counters[C8OPT_CNT_INVALID] = cnt[6];
        counters[C8OPT_CNT_CULLED] = cnt[7];
    }
    if (dropped) return fail(ctx, C8OPT_ERR_CAPACITY, "%llu photon records dropped: output capacity exceeded", dropped);
    return C8OPT_OK;
}

int c8opt_reset_tallies(c8opt_ctx *ctx, void *cuda_stream)
{
    if (!ctx) return C8OPT_ERR_ARGUMENT;
    DeviceGuard guard(ctx->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    C8_CUDA(ctx, cudaMemsetAsync(ctx->d_results, 0, 64 + 32 * (size_t)ctx->n_tel, st));      // counters, cursors, tallies
    if (ctx->d_hist) C8_CUDA(ctx, cudaMemsetAsync(ctx->d_hist, 0, sizeof(c8::Tally) * (ctx->hist_bins + 1), st));
    ctx->segments_total = 0;
    return C8OPT_OK;
}

int c8opt_set_ground_histogram(c8opt_ctx *ctx, double core_x_m, double core_y_m, double r_max_m, int32_t n_bins)
{
    if (!ctx) return C8OPT_ERR_ARGUMENT;
    if (n_bins < 0 || n_bins > c8::kHistMax) return fail(ctx, C8OPT_ERR_ARGUMENT, "n_bins must be 0 .. %d", c8::kHistMax);
    if (n_bins > 0 && (!std::isfinite(core_x_m) || !std::isfinite(core_y_m) || !(r_max_m > 0.0) || !std::isfinite(r_max_m)))
        return fail(ctx, C8OPT_ERR_ARGUMENT, "need a finite core and r_max > 0");
    DeviceGuard guard(ctx->device);
    C8_CUDA(ctx, cudaDeviceSynchronize());
    cudaFree(ctx->d_hist);
    ctx->d_hist = nullptr; ctx->hist_bins = 0;
    if (n_bins == 0) return C8OPT_OK;
    C8_CUDA(ctx, cudaMalloc(&ctx->d_hist, sizeof(c8::Tally) * (n_bins + 1)));
    C8_CUDA(ctx, cudaMemset(ctx->d_hist, 0, sizeof(c8::Tally) * (n_bins + 1)));
    ctx->hist_bins = n_bins; ctx->hist_core_x = core_x_m; ctx->hist_core_y = core_y_m; ctx->hist_r_max = r_max_m;
    return C8OPT_OK;
}

int c8opt_read_ground_histogram(c8opt_ctx *ctx, c8opt_hist_bin *host_out, int32_t n_bins, uint64_t *overflow, uint64_t *counters)
{
    if (!ctx) return C8OPT_ERR_ARGUMENT;
    if (!host_out) return fail(ctx, C8OPT_ERR_ARGUMENT, "host_out is NULL");
    if (n_bins != ctx->hist_bins || n_bins < 1) return fail(ctx, C8OPT_ERR_ARGUMENT, "n_bins = %d but the context has %d bins", n_bins, ctx->hist_bins);
    DeviceGuard guard(ctx->device);
    C8_CUDA(ctx, cudaDeviceSynchronize());
    static_assert(sizeof(c8opt_hist_bin) == sizeof(c8::Tally), "histogram bin layout");
    C8_CUDA(ctx, cudaMemcpy(host_out, ctx->d_hist, sizeof(c8::Tally) * n_bins, cudaMemcpyDeviceToHost));
    c8::Tally over;
    C8_CUDA(ctx, cudaMemcpy(&over, ctx->d_hist + n_bins, sizeof(over), cudaMemcpyDeviceToHost));
    if (overflow) *overflow = over.hits;
    if (counters) {
        unsigned long long cnt[8];
        C8_CUDA(ctx, cudaMemcpy(cnt, ctx->d_counters, sizeof(cnt), cudaMemcpyDeviceToHost));
        unsigned long long inside = 0;
        for (int b = 0; b < n_bins; ++b) inside += host_out[b].n;
        counters[C8OPT_CNT_SEGMENTS] = ctx->segments_total;
        counters[C8OPT_CNT_GENERATED] = cnt[1];
        counters[C8OPT_CNT_UPWARD] = cnt[2];
        counters[C8OPT_CNT_HITS] = inside + over.hits;
        counters[C8OPT_CNT_RECORDS] = 0;
        counters[C8OPT_CNT_DROPPED] = 0;
        counters[C8OPT_CNT_INVALID] = cnt[6];
        counters[C8OPT_CNT_CULLED] = cnt[7];
    }
    return C8OPT_OK;
}

void c8opt_destroy(c8opt_ctx *ctx)
{
    if (!ctx) return;
    DeviceGuard guard(ctx->device);
    cudaDeviceSynchronize();
    for (int i = 0; i < c8opt_ctx::kPipe; ++i) {
        if (ctx->pipe_stream[i]) cudaStreamDestroy(ctx->pipe_stream[i]);
        cudaFree(ctx->d_stage[i]);
    }
    for (int i = 0; i <= c8opt_ctx::kPipe; ++i) if (ctx->pipe_event[i]) cudaEventDestroy(ctx->pipe_event[i]);
    cudaFree(ctx->d_telD);
    cudaFree(ctx->d_tau); cudaFree(ctx->d_telA); cudaFree(ctx->d_telT); cudaFree(ctx->d_telEta); cudaFree(ctx->d_grid);
    cudaFree(ctx->d_results); cudaFreeHost(ctx->h_results); cudaFree(ctx->d_hist);
    cudaGetLastError();
    delete ctx;
}

const char *c8opt_last_error(const c8opt_ctx *ctx) { return ctx ? ctx->error : g_create_error; }

uint64_t c8opt_launch_count(const c8opt_ctx *ctx) { return ctx ? ctx->launches : 0; }

}  // extern "C"

// ------------------------------------------------------------------------------------------------------------------
// c8opt_tally_static: the tally pass with no context and no allocation (include/c8opt.h).  Everything the context
// path keeps in cudaMalloc'ed memory sits in this one array; host code must not pass its NAME to a kernel (that is a
// host-side stand-in): static_device() asks for the device address once per device, kernels in this file name it
// directly.
// Layout: [0, 384) the result block of 8 telescopes as in c8opt_ctx (counters 8 x u64, cursors, tallies, capacities);
// [512, 640) telA float4[8]; [640, 672) telT; [672, 704) telEta; [704, 960) telD double4[8].
static __device__ __align__(256) unsigned char g_c8opt_static_scratch[C8OPT_STATIC_SCRATCH_BYTES];

namespace {

constexpr int kStaticTel = C8OPT_STATIC_MAX_TELESCOPES;
static_assert(kStaticTel == c8::kTelConstMax, "the static entry point serves the brute-force kernels (telescopes in the constant bank)");
constexpr size_t kStOffCursors = 64, kStOffTallies = 64 + 8 * kStaticTel, kStOffTelA = 512, kStOffTelT = 640,
                 kStOffTelEta = 672, kStOffTelD = 704;
static_assert(kStOffTallies + (sizeof(c8::Tally) + 8) * kStaticTel <= kStOffTelA, "result block overlaps the tables");
static_assert(kStOffTelD + sizeof(double4) * kStaticTel <= C8OPT_STATIC_SCRATCH_BYTES, "static scratch too small");

struct StaticTables { float4 telA[kStaticTel]; double4 telD[kStaticTel]; float telT[kStaticTel], telEta[kStaticTel]; };

// Writes the telescope tables and zeroes the accumulators (the array keeps the last call's contents).
__global__ void static_setup_kernel(const StaticTables t)
{
    unsigned char *s = g_c8opt_static_scratch;
    const int i = threadIdx.x;
    if (i < (int)(kStOffTelA / 8)) reinterpret_cast<unsigned long long *>(s)[i] = 0ull;
    if (i < kStaticTel) {
        reinterpret_cast<float4 *>(s + kStOffTelA)[i] = t.telA[i];
        reinterpret_cast<float *>(s + kStOffTelT)[i] = t.telT[i];
        reinterpret_cast<float *>(s + kStOffTelEta)[i] = t.telEta[i];
        reinterpret_cast<double4 *>(s + kStOffTelD)[i] = t.telD[i];
    }
}

// Results to the caller's buffers: the tallies, and the counters in the order of C8OPT_CNT_*.
__global__ void static_finish_kernel(c8::Tally *tallies_out, unsigned long long *counters_out, int n_tel, unsigned long long n_seg)
{
    const unsigned char *s = g_c8opt_static_scratch;
    const c8::Tally *t = reinterpret_cast<const c8::Tally *>(s + kStOffTallies);
    const int i = threadIdx.x;
    if (i < n_tel) tallies_out[i] = t[i];
    if (i == 0 && counters_out) {
        const unsigned long long *cnt = reinterpret_cast<const unsigned long long *>(s);
        unsigned long long hits = 0;
        for (int k = 0; k < n_tel; ++k) hits += t[k].hits;
        counters_out[C8OPT_CNT_SEGMENTS] = n_seg; counters_out[C8OPT_CNT_GENERATED] = cnt[1];
        counters_out[C8OPT_CNT_UPWARD] = cnt[2]; counters_out[C8OPT_CNT_HITS] = hits;
        counters_out[C8OPT_CNT_RECORDS] = 0; counters_out[C8OPT_CNT_DROPPED] = 0;
        counters_out[C8OPT_CNT_INVALID] = cnt[6]; counters_out[C8OPT_CNT_CULLED] = cnt[7];
    }
}

// Once per device, with that device current: the array's device address, the SM count, the shared-memory limit of the
// six brute-force tally kernels.  No allocation.
struct StaticDevice { bool ready = false; unsigned char *scratch = nullptr; int n_sm = 148; };
constexpr int kStaticDevices = 64;
StaticDevice g_static_device[kStaticDevices];
std::mutex g_static_mutex;

int static_device(int dev, StaticDevice *out)
{
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticDevice &d = g_static_device[dev];
    if (!d.ready) {
        int major = 0, n_sm = 0;
        C8_CUDA(nullptr, cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
        if (major != 10) return fail(nullptr, C8OPT_ERR_CUDA, "device is sm_%dx, this library is built for sm_100a only", major);
        C8_CUDA(nullptr, cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
        unsigned char *ptr = nullptr;
        C8_CUDA(nullptr, cudaGetSymbolAddress((void **)&ptr, g_c8opt_static_scratch));
        if (!ptr) return fail(nullptr, C8OPT_ERR_CUDA, "cudaGetSymbolAddress gave no address for the static scratch");
        for (int nt = 1; nt <= 8; nt *= (nt == 1 ? 4 : 2))
            for (int cp = 0; cp < 2; ++cp)
                C8_CUDA(nullptr, cudaFuncSetAttribute(pick_kernel(c8::TEL_CONST, cp != 0, nt, 0), cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                      (int)smem_bytes(c8::MODE_TALLY)));
        C8_CUDA(nullptr, cudaFuncSetAttribute(pick_disp_kernel(c8::TEL_CONST, 0), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes(c8::MODE_TALLY)));
        d.scratch = ptr; d.n_sm = n_sm > 0 ? n_sm : 148; d.ready = true;
    }
    *out = d;
    return C8OPT_OK;
}

}  // namespace

extern "C" int c8opt_tally_static(const c8opt_atmosphere_desc *desc, const float *d_tau, const float *xyzr, int32_t n_tel,
                                  const c8opt_segment *d_seg, uint64_t n, uint64_t first_segment_id,
                                  const c8opt_run_params *params, c8opt_tally *d_tallies_out, uint64_t *d_counters_out,
                                  void *cuda_stream)
{
    if (!desc || !xyzr || !params || !d_tallies_out) return fail(nullptr, C8OPT_ERR_ARGUMENT, "c8opt_tally_static: atmosphere, xyzr, params or d_tallies_out is NULL");
    if (!d_seg && n) return fail(nullptr, C8OPT_ERR_ARGUMENT, "c8opt_tally_static: d_seg is NULL");
    if (n_tel < 1) return fail(nullptr, C8OPT_ERR_ARGUMENT, "c8opt_tally_static: telescope count %d must be >= 1", n_tel);
    if (n_tel > kStaticTel)
        return fail(nullptr, C8OPT_ERR_ARGUMENT, "c8opt_tally_static: %d telescopes, but the static scratch (%d bytes) holds the tables and "
                    "accumulators of at most %d: use a context (c8opt_create_atmosphere)", n_tel, C8OPT_STATIC_SCRATCH_BYTES, kStaticTel);
    if (params->mode != C8OPT_MODE_TALLY) return fail(nullptr, C8OPT_ERR_ARGUMENT, "c8opt_tally_static: mode must be C8OPT_MODE_TALLY");
    if (desc->n_layers < 1 || desc->n_layers > C8OPT_MAX_LAYERS) return fail(nullptr, C8OPT_ERR_ARGUMENT, "n_layers out of range");
    for (int i = 0; i < desc->n_layers; ++i) {
        const c8opt_layer &l = desc->layers[i];
        if (!std::isfinite(l.h_lo_m) || !std::isfinite(l.a_gcm2) || !std::isfinite(l.b_gcm2) || !(l.c_m > 0.0) || !std::isfinite(l.c_m))
            return fail(nullptr, C8OPT_ERR_ARGUMENT, "layer %d: non-finite coefficient or c <= 0", i);
        if (i > 0 && !(l.h_lo_m > desc->layers[i - 1].h_lo_m)) return fail(nullptr, C8OPT_ERR_ARGUMENT, "layer bounds must ascend");
    }
    if (!(desc->rho0_gcm3 > 0.0) || !std::isfinite(desc->eta0) || !(desc->eta0 >= 0.0) || !std::isfinite(desc->h_obs_m))
        return fail(nullptr, C8OPT_ERR_ARGUMENT, "need rho0 > 0, eta0 >= 0, finite h_obs");
    if (d_tau && (desc->tau_nh < 1 || desc->tau_nl < 1 || desc->tau_nh > 4096 || desc->tau_nl > 4096 || !(desc->tau_dh_m > 0.0) || !(desc->tau_dl_nm > 0.0)))
        return fail(nullptr, C8OPT_ERR_ARGUMENT, "bad transmission table shape / spacing");
    for (int k = 0; k < n_tel; ++k) {
        for (int i = 0; i < 4; ++i)
            if (!std::isfinite(xyzr[4 * k + i])) return fail(nullptr, C8OPT_ERR_ARGUMENT, "telescope %d: non-finite value", k);
        if (!(xyzr[4 * k + 3] > 0.0f)) return fail(nullptr, C8OPT_ERR_ARGUMENT, "telescope %d: radius must be > 0", k);
    }
    int ndev = 0, dev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(nullptr, C8OPT_ERR_CUDA, "no CUDA device (this library has no CPU fallback)");
    }
    C8_CUDA(nullptr, cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticDevices) return fail(nullptr, C8OPT_ERR_CUDA, "device ordinal %d out of range", dev);
    StaticDevice sd;
    int rc = static_device(dev, &sd);
    if (rc != C8OPT_OK) return rc;

    // Host-side description of the run (what c8opt_create_atmosphere and c8opt_add_telescopes keep in a context), with
    // the device pointers aimed at the static array.  Per thread; its small host vectors are sized on the first call.
    thread_local c8opt_ctx host;
    c8opt_ctx *ctx = &host;
    ctx->device = dev; ctx->n_sm = sd.n_sm;
    ctx->n_layers = desc->n_layers;
    for (int i = 0; i < desc->n_layers; ++i)
        ctx->layer[i] = HostLayer{desc->layers[i].h_lo_m, desc->layers[i].a_gcm2, desc->layers[i].b_gcm2, desc->layers[i].c_m};
    ctx->eta0 = desc->eta0; ctx->rho0 = desc->rho0_gcm3; ctx->h_obs = desc->h_obs_m;
    ctx->d_tau = const_cast<float *>(d_tau);
    ctx->tau_nh = d_tau ? desc->tau_nh : 0; ctx->tau_nl = d_tau ? desc->tau_nl : 0;
    ctx->tau_h0 = d_tau ? desc->tau_h0_m : 0.0; ctx->tau_dh = d_tau ? desc->tau_dh_m : 1.0;
    ctx->tau_l0 = d_tau ? desc->tau_l0_nm : 0.0; ctx->tau_dl = d_tau ? desc->tau_dl_nm : 1.0;
    // telescopes: the host part of c8opt_add_telescopes
    double lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    for (int k = 0; k < n_tel; ++k)
        for (int i = 0; i < 3; ++i) { lo[i] = std::fmin(lo[i], xyzr[4 * k + i]); hi[i] = std::fmax(hi[i], xyzr[4 * k + i]); }
    ctx->tel_xyzr.assign(xyzr, xyzr + 4 * (size_t)n_tel);
    ctx->x_ref = 0.5 * (lo[0] + hi[0]); ctx->y_ref = 0.5 * (lo[1] + hi[1]); ctx->z_ref = 0.5 * (lo[2] + hi[2]);
    ctx->coplanar = (lo[2] == hi[2]);
    ctx->h_telA.resize(n_tel); ctx->h_telT.resize(n_tel); ctx->h_telEta.resize(n_tel);
    StaticTables tab;
    std::memset(&tab, 0, sizeof(tab));
    double z_low = INFINITY, rb = 0.0;
    ctx->r_max = 0.0;
    for (int k = 0; k < n_tel; ++k) {
        const double x = xyzr[4 * k], y = xyzr[4 * k + 1], z = xyzr[4 * k + 2], r = xyzr[4 * k + 3];
        ctx->h_telA[k] = make_float4((float)(x - ctx->x_ref), (float)(y - ctx->y_ref), (float)(z - ctx->z_ref), (float)(r * r));
        ctx->h_telT[k] = (float)host_depth(ctx, z);
        ctx->h_telEta[k] = (float)host_refractivity(ctx, z);
        z_low = std::fmin(z_low, z); ctx->r_max = std::fmax(ctx->r_max, r);
        const double dx = x - ctx->x_ref, dy = y - ctx->y_ref, dz = z - ctx->z_ref;
        rb = std::fmax(rb, std::sqrt(dx * dx + dy * dy + dz * dz) + r);
        tab.telA[k] = ctx->h_telA[k]; tab.telT[k] = ctx->h_telT[k]; tab.telEta[k] = ctx->h_telEta[k];
        tab.telD[k] = make_double4(x, y, z, r);
    }
    ctx->refr_cmax = 0.01 * ctx->eta0 / ctx->rho0 * host_depth(ctx, z_low);
    ctx->cull_Rb = (float)(rb * (1.0 + 1e-6));
    ctx->array_rb = rb;
    ctx->tel_src = c8::TEL_CONST; ctx->n_tel = n_tel; ctx->n_grid_levels = 0; ctx->d_grid = nullptr; ctx->have_refract_grid = false;
    ctx->d_results = sd.scratch;
    ctx->d_counters = reinterpret_cast<unsigned long long *>(sd.scratch);
    ctx->d_cursors = reinterpret_cast<unsigned long long *>(sd.scratch + kStOffCursors);
    ctx->d_tallies = reinterpret_cast<c8::Tally *>(sd.scratch + kStOffTallies);
    ctx->d_telA = reinterpret_cast<float4 *>(sd.scratch + kStOffTelA);
    ctx->d_telT = reinterpret_cast<float *>(sd.scratch + kStOffTelT);
    ctx->d_telEta = reinterpret_cast<float *>(sd.scratch + kStOffTelEta);
    ctx->d_telD = reinterpret_cast<double4 *>(sd.scratch + kStOffTelD);

    c8::KParams P;
    rc = fill_params(ctx, params, nullptr, &P);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (rc == C8OPT_OK) {
        static_setup_kernel<<<1, 64, 0, st>>>(tab);
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) rc = fail(ctx, C8OPT_ERR_CUDA, "static_setup_kernel: %s", cudaGetErrorString(e));
    }
    if (rc == C8OPT_OK) rc = launch(ctx, P, params->mode, d_seg, n, first_segment_id, nullptr, st);
    if (rc == C8OPT_OK) {
        static_finish_kernel<<<1, 32, 0, st>>>(reinterpret_cast<c8::Tally *>(d_tallies_out),
                                              reinterpret_cast<unsigned long long *>(d_counters_out), n_tel, n);
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) rc = fail(ctx, C8OPT_ERR_CUDA, "static_finish_kernel: %s", cudaGetErrorString(e));
    }
    // the thread's host object must not own (and its destructor does not touch) the static array or the caller's table
    ctx->d_results = nullptr; ctx->d_tau = nullptr; ctx->d_telA = nullptr; ctx->d_telT = nullptr; ctx->d_telEta = nullptr; ctx->d_telD = nullptr;
    if (rc != C8OPT_OK) { std::memcpy(g_create_error, ctx->error, sizeof(g_create_error)); g_create_error[255] = 0; }
    return rc;
}
