// modal_api.cu -- the C ABI of include/modal.h: plan, coefficient upload, launch logic.
// Host-side derivations live in host_math.hpp, kernels in kernels.cuh.
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <numeric>
#include <string>
#include <vector>

#include "../../include/modal.h"
#include "host_math.hpp"
#include "flow_schedule.hpp"
#include "mma_schedule.hpp"
#include "stream_schedule.hpp"
#include "kernels.cuh"
#include "vk_flow.cuh"
#include "vk_mma.cuh"
#include "vk_stream.cuh"
#include "vk_bptt.cuh"
#include "vk_small.cuh"
#include "vk_dense.cuh"
#include "vk_repl.cuh"
#include "repl_schedule.hpp"
#include "peaks.cuh"

namespace mh = modal_host;
namespace md = modal_dev;

static_assert(mh::MMA_RB_MAX == md::MMA_RB_MAX_DEV && mh::MMA_NG_MAX == md::MMA_NG_MAX_DEV && mh::MMA_MT_MAX == md::MMA_MT_MAX &&
              mh::MMA_FBLK_MAX == 16 && mh::MMA_KCL_MAX == 64, "batched-kernel limits");

namespace {

thread_local std::string g_create_error;   // messages of a failed modal_plan_create

constexpr size_t SMEM_LIMIT = 227 * 1024;  // opt-in dynamic shared memory per CTA on sm_100

struct DevBuf {
    void *p = nullptr; size_t bytes = 0;
    cudaError_t ensure(size_t n) {
        if (n <= bytes) return cudaSuccess;
        if (p) cudaFree(p);
        p = nullptr; bytes = 0;
        cudaError_t e = cudaMalloc(&p, n);
        if (e == cudaSuccess) bytes = n;
        return e;
    }
    void release() { if (p) cudaFree(p); p = nullptr; bytes = 0; }
    template <class T> T *as() const { return reinterpret_cast<T *>(p); }
};

struct FlowConfig {
    int G = 1, NT = 1, NW = 16, NS = 0, slot_tiles = 8, res_tiles = 0, direct = 0, streamed = 0;
    size_t smem = 0;
    mh::FlowSchedule sched;
    DevBuf dsched;
    bool uploaded = false;
};

struct MmaConfig {
    bool tried = false, ok = false;
    mh::MmaLayout L;
    int lpq = 1;                     // lanes of an owner team that share one quad of the partial-force gather
    size_t off_nlist = 0, off_klist = 0, off_kcnt = 0, off_fblk = 0, off_fcnt = 0, off_blk = 0;   // ints into dtab
    DevBuf dslabs, dtab, dQop, dqf, dGx, dfx, dflags, dpx;
};

struct ReplConfig {                  // vk_repl: replicated state, whole in-plane modes per CTA (one sample)
    bool tried = false, ok = false;
    int CL = 1, NCL = 1, SL = 0, NQ2 = 0;
    size_t smem = 0;
    mh::ReplLayout L;
    DevBuf dHp, dtab, dcls, dX;
};

struct StreamConfig {                // vk_stream: layout for one NB (samples of a launch, padded to 16)
    bool ok = false;
    int NB = 0, lpq = 1;
    mh::StreamLayout L;
    size_t off_cta = 0, off_tile = 0, off_blk = 0, off_nct = 0;
    DevBuf dA, dtab, dqx, dGx, dfx, dpx;
};

struct Options {                     // modal_plan_set_option
    int vk_impl = 0, flow_g = 0, flow_ns = 0, flow_res = -1, mma_split = 0, mma_ng = 0, mma_nstg = 0, mma_cluster = 1, parity_order = 1, timing = 0;
};

}  // namespace

struct modal_plan {
    modal_plan_desc d{};
    int device = -1;
    double T = 0;
    mh::ModeSet mq, mphi;
    int NQP = 0;                 // padded mode count of the device layout
    int coeff_batch = 1;
    std::vector<double> omega, sigma, nl_scale, lambda_s, pickup;   // [coeff_batch][...]
    std::vector<int> active;                                          // [coeff_batch][n_q]
    std::vector<float> Hf;                                            // flow-tile-packed H (VK, flow kernel), INTERNAL mode order
    std::vector<uint8_t> tile_nz;                                     // per flow tile: holds a non-zero entry
    long long nz_tiles = 0;
    // internal (device) order of the transverse modes: perm[k_internal] = k_user.  VK plates group the modes by index
    // parity (m mod 2, n mod 2): H^n couples only parity classes c and c xor delta_n, so whole 16x16 tiles vanish.
    std::vector<int> perm, iperm;
    int airy_basis = 0;                                               // modal_airy_basis
    std::vector<double> zeta4;                                        // [n_phi] of the reference geometry
    bool coeffs_dirty = true, H_dirty = true;
    std::string err;
    int sm_count = 148;
    // device storage
    DevBuf dHf, dfx, dgx, dqx, dtiming, dperm, dtimeout;
    MmaConfig mma;
    StreamConfig stream;
    DevBuf bp[16];                                                    // modal_bptt: dense H, coefficients, gradients, scratch
    bool bp_H_valid = false;
    DevBuf dHdense, ddscr; bool dense_H_valid = false;                // vk_dense_kernel: dense fp32 H (internal order, padded rows), exchange words
    DevBuf dHsmall; bool small_H_valid = false;                       // vk_small_kernel: dense fp32 H, internal order
    ReplConfig repl;
    std::map<long long, FlowConfig> flow_cfgs;
    DevBuf dkv, dkq, dr, dast, ds, dsT, dw, dlam, dc, dq0, dv0, dgain, dbad, dout;      // dsT: s_n transposed [n_phi][coeff_batch] (batched kernel)
    float *pinned_out = nullptr; size_t pinned_bytes = 0;            // staging of modal_simulate_host
    Options opt;
    int kinfo[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    // the last modal_simulate call (modal_plan_check)
    cudaStream_t last_stream = nullptr; int last_batch = 0; bool last_persistent = false, pending = false;
};

namespace {

#define CU(call)                                                                             \
    do {                                                                                     \
        cudaError_t e_ = (call);                                                             \
        if (e_ != cudaSuccess) {                                                             \
            p->err += std::string("CUDA error: ") + cudaGetErrorString(e_) + " at " #call "\n"; \
            return MODAL_ECUDA;                                                              \
        }                                                                                    \
    } while (0)

int n_nl(const modal_plan *p) { return p->d.model == MODAL_VK ? p->d.n_phi : 1; }

// Internal order of the transverse modes (see modal_plan::perm).
void build_perm(modal_plan *p)
{
    const int nq = p->d.n_q;
    p->perm.resize(nq); p->iperm.resize(nq);
    for (int k = 0; k < nq; ++k) p->perm[k] = k;
    if (p->d.model == MODAL_VK && p->d.geom == MODAL_RECT && p->opt.parity_order)
        std::stable_sort(p->perm.begin(), p->perm.end(), [&](int a, int b) {
            return ((p->mq.m[a] & 1) * 2 + (p->mq.n[a] & 1)) < ((p->mq.m[b] & 1) * 2 + (p->mq.n[b] & 1));
        });
    for (int k = 0; k < nq; ++k) p->iperm[p->perm[k]] = k;
}

// Store H (given in USER mode order) as flow tiles in internal order; note which tiles are entirely zero.
template <class Get>
void set_H(modal_plan *p, Get get_user)
{
    const int nq = p->d.n_q, nphi = p->d.n_phi;
    auto get = [&](int n, int a, int b) { return get_user(n, p->perm[a], p->perm[b]); };
    mh::pack_flow_tiles(nq, nphi, get, p->Hf);
    const size_t ntiles = p->Hf.size() / mh::FT_FLOATS;
    p->tile_nz.assign(ntiles, 0);
    p->nz_tiles = 0;
    for (size_t t = 0; t < ntiles; ++t) {
        const float *x = &p->Hf[t * mh::FT_FLOATS];
        uint8_t nz = 0;
        for (int e = 0; e < mh::FT_FLOATS; ++e) if (x[e] != 0.f) { nz = 1; break; }
        p->tile_nz[t] = nz; p->nz_tiles += nz;
    }
    for (auto &kv : p->flow_cfgs) kv.second.dsched.release();
    p->flow_cfgs.clear();                                   // schedules depend on the zero pattern
    p->mma.tried = false; p->mma.ok = false; p->repl.tried = false; p->repl.ok = false; p->stream.NB = 0; p->bp_H_valid = false; p->small_H_valid = false; p->dense_H_valid = false;
    p->H_dirty = true;
}

bool validate_desc(const modal_plan_desc &d, std::string &err)
{
    auto bad = [&](const char *m) { err += m; err += "\n"; };
    if (d.model < MODAL_LINEAR || d.model > MODAL_VK) bad("model must be MODAL_LINEAR, MODAL_TENSION or MODAL_VK");
    if (d.scheme != MODAL_SV && d.scheme != MODAL_FTM) bad("scheme must be MODAL_SV or MODAL_FTM");
    if (d.geom != MODAL_STRING && d.geom != MODAL_RECT) bad("geom must be MODAL_STRING or MODAL_RECT");
    if (d.bc != MODAL_BC_FIXED_SS) bad("bc must be MODAL_BC_FIXED_SS");
    if (d.model == MODAL_VK && d.geom != MODAL_RECT) bad("MODAL_VK needs MODAL_RECT geometry");
    if (!(d.Lx > 0)) bad("Lx must be positive");
    if (d.geom == MODAL_RECT && !(d.Ly > 0)) bad("Ly must be positive");
    if (d.geom == MODAL_RECT && !(d.h > 0)) bad("h must be positive");
    if (!(d.rho > 0)) bad("rho must be positive");
    if (!(d.E >= 0)) bad("E must be non-negative");
    if (d.geom == MODAL_RECT && !(d.nu > -1.0 && d.nu < 0.5 + 1e-12)) bad("nu must lie in (-1, 0.5]");
    if (!(d.T0 >= 0)) bad("T0 must be non-negative");
    if (d.geom == MODAL_STRING && !(d.T0 > 0) && !(d.D > 0)) bad("degenerate dispersion: T0 and D both zero");
    if (!(d.sigma0 >= 0) || !(d.sigma1 >= 0)) bad("sigma0 and sigma1 must be non-negative");
    if (d.n_q < 1) bad("n_q must be at least 1");
    if (d.model == MODAL_VK && d.n_phi < 1) bad("MODAL_VK needs n_phi >= 1");
    if (d.model != MODAL_VK && d.n_phi != 0) bad("n_phi must be 0 unless MODAL_VK");
    if (!(d.sample_rate > 0)) bad("sample_rate must be positive");
    if (d.max_batch < 1) bad("max_batch must be at least 1");
    if (d.max_steps < 1) bad("max_steps must be at least 1");
    if (d.geom == MODAL_RECT) {
        if (!(d.pickup_x >= 0 && d.pickup_x <= d.Lx) || !(d.pickup_y >= 0 && d.pickup_y <= d.Ly))
            bad("pickup point must lie on the plate");
    } else if (!(d.pickup_x >= 0 && d.pickup_x <= d.Lx)) bad("pickup point must lie on the string");
    return err.empty();
}

double mode_value(const modal_plan *p, int k, double Lx, double Ly, double x, double y)
{
    if (p->d.geom == MODAL_STRING) return std::sqrt(2.0 / Lx) * std::sin(p->mq.m[k] * mh::PI * x / Lx);
    return 2.0 / std::sqrt(Lx * Ly) * std::sin(p->mq.m[k] * mh::PI * x / Lx) * std::sin(p->mq.n[k] * mh::PI * y / Ly);
}

// Fill one row of per-sample coefficients for a geometry (plan index sets).
void derive_row(const modal_plan *p, const modal_sample_geom &g, double *omega, double *sigma,
                double *nl_scale, double *lambda, double *pickup)
{
    const modal_plan_desc &d = p->d;
    const int nq = d.n_q;
    std::vector<double> lam(nq);
    if (d.geom == MODAL_RECT) {
        for (int k = 0; k < nq; ++k) lam[k] = mh::rect_lambda(p->mq.m[k], p->mq.n[k], g.Lx, g.Ly);
        const double D = (d.D > 0 && g.h == d.h) ? d.D : mh::plate_D(d.E, g.h, d.nu);
        mh::omega_sigma(lam, D, d.T0, d.rho * g.h, d.sigma0, d.sigma1, omega, sigma);   // reading R3: rho h
        if (d.model == MODAL_VK && nl_scale) {
            const double cb = std::pow(g.Lx * g.Ly, -2.5), cref = std::pow(d.Lx * d.Ly, -2.5);
            for (int n = 0; n < d.n_phi; ++n) {
                const double z = mh::rect_lambda(p->mphi.m[n], p->mphi.n[n], g.Lx, g.Ly);   // zeta^4 = lambda^2 (R5)
                nl_scale[n] = d.E / (2.0 * d.rho * z * z) * (cb / cref) * (cb / cref);       // reading R14
            }
        } else if (d.model == MODAL_TENSION && nl_scale) {
            nl_scale[0] = d.E * g.h / (2.0 * g.Lx * g.Ly * (1.0 - d.nu * d.nu)) / (d.rho * g.h);   // Berger, Eq. 4
        } else if (nl_scale) nl_scale[0] = 0.0;
        if (pickup)
            for (int k = 0; k < nq; ++k)
                pickup[k] = mode_value(p, k, g.Lx, g.Ly, g.pickup_x_frac * g.Lx, g.pickup_y_frac * g.Ly);
    } else {
        for (int k = 0; k < nq; ++k) lam[k] = (p->mq.m[k] * mh::PI / g.Lx) * (p->mq.m[k] * mh::PI / g.Lx);
        mh::omega_sigma(lam, g.D, g.T0, g.rho, d.sigma0, d.sigma1, omega, sigma);
        if (nl_scale) nl_scale[0] = d.model == MODAL_TENSION ? d.E * g.area / (2.0 * g.Lx) / g.rho : 0.0;   // Eq. 4
        if (pickup)
            for (int k = 0; k < nq; ++k) pickup[k] = mode_value(p, k, g.Lx, 0, g.pickup_x_frac * g.Lx, 0);
    }
    if (lambda) for (int k = 0; k < nq; ++k) lambda[k] = lam[k];
}

modal_sample_geom fill_geom(const modal_plan *p, const modal_sample_geom *in)
{
    const modal_plan_desc &d = p->d;
    modal_sample_geom g{};
    auto pick = [](double v, double def) { return (v > 0) ? v : def; };
    g.Lx = pick(in ? in->Lx : 0, d.Lx); g.Ly = pick(in ? in->Ly : 0, d.Ly); g.h = pick(in ? in->h : 0, d.h);
    g.T0 = pick(in ? in->T0 : 0, d.T0); g.D = pick(in ? in->D : 0, d.D); g.rho = pick(in ? in->rho : 0, d.rho);
    g.area = pick(in ? in->area : 0, d.area);
    g.pickup_x_frac = (in && in->pickup_x_frac > 0) ? in->pickup_x_frac : d.pickup_x / d.Lx;
    g.pickup_y_frac = (in && in->pickup_y_frac > 0) ? in->pickup_y_frac
                                                    : (d.geom == MODAL_RECT ? d.pickup_y / d.Ly : 0.0);
    return g;
}

// Recompute masks and delta-form coefficients from (omega, sigma, ...) and upload them.
modal_status sync_coeffs(modal_plan *p)
{
    const modal_plan_desc &d = p->d;
    const int cb = p->coeff_batch, nq = d.n_q, P = p->NQP, nnl = n_nl(p);
    p->active.assign((size_t)cb * nq, 0);
    std::vector<double> kv((size_t)cb * P, 0.0), kq(kv), r(kv), ast(kv);
    std::vector<float> w((size_t)cb * P, 0.f), lam((size_t)cb * P, 0.f), s((size_t)cb * nnl, 0.f);
    int masked = 0;
    for (int b = 0; b < cb; ++b)
        for (int k = 0; k < nq; ++k) {
            const double om = p->omega[(size_t)b * nq + k], sg = p->sigma[(size_t)b * nq + k];
            const bool act = mh::mode_active(d.scheme, om, sg, p->T) && std::isfinite(om) && std::isfinite(sg);
            p->active[(size_t)b * nq + k] = act;
            if (!act) { ++masked; continue; }
            if (d.scheme == MODAL_FTM && !(om > sg)) {        // the FTM coefficients need an underdamped mode
                char buf[200];
                snprintf(buf, sizeof buf, "FTM scheme: mode %d of coefficient row %d is critically damped or overdamped "
                         "(omega = %.6g <= sigma = %.6g)\n", k, b, om, sg);
                p->err += buf;
                return MODAL_EINVAL;
            }
            const mh::StepCoeffs c = mh::step_coeffs(d.scheme, om, sg, p->T);
            const size_t o = (size_t)b * P + p->iperm[k];
            kv[o] = c.kv; kq[o] = c.kq; r[o] = c.r; ast[o] = c.astart;
            w[o] = (float)p->pickup[(size_t)b * nq + k];
            if (d.model != MODAL_VK) lam[o] = (float)p->lambda_s[(size_t)b * nq + k];
        }
    for (size_t i = 0; i < s.size(); ++i) s[i] = (float)p->nl_scale[i];
    if (masked) {
        char buf[160];
        snprintf(buf, sizeof buf, "warning: %d mode-rows masked (beyond the stability limit of the scheme, reading R11)\n", masked);
        p->err += buf;
    }
    if (p->device < 0) { p->coeffs_dirty = false; return MODAL_OK; }
    CU(cudaSetDevice(p->device));
    auto up = [&](DevBuf &b, const void *src, size_t bytes) -> cudaError_t {
        cudaError_t e = b.ensure(bytes);
        if (e != cudaSuccess) return e;
        return cudaMemcpy(b.p, src, bytes, cudaMemcpyHostToDevice);
    };
    CU(up(p->dkv, kv.data(), kv.size() * 8)); CU(up(p->dkq, kq.data(), kq.size() * 8));
    CU(up(p->dr, r.data(), r.size() * 8));    CU(up(p->dast, ast.data(), ast.size() * 8));
    CU(up(p->dw, w.data(), w.size() * 4));
    if (d.model == MODAL_VK) {
        CU(up(p->ds, s.data(), s.size() * 4));
        std::vector<float> sT(s.size());                          // [n_phi][cb]: consecutive samples read consecutive words
        for (int b = 0; b < cb; ++b) for (int n = 0; n < nnl; ++n) sT[(size_t)n * cb + b] = s[(size_t)b * nnl + n];
        CU(up(p->dsT, sT.data(), sT.size() * 4));
    }
    else { CU(up(p->dlam, lam.data(), lam.size() * 4)); CU(up(p->dc, s.data(), s.size() * 4)); }
    p->coeffs_dirty = false;
    return MODAL_OK;
}

modal_status sync_H(modal_plan *p)
{
    if (p->device >= 0 && p->d.model == MODAL_VK) {
        CU(cudaSetDevice(p->device));
        CU(p->dHf.ensure(p->Hf.size() * 4));
        CU(cudaMemcpy(p->dHf.p, p->Hf.data(), p->Hf.size() * 4, cudaMemcpyHostToDevice));
        CU(p->dperm.ensure(p->perm.size() * 4));
        CU(cudaMemcpy(p->dperm.p, p->perm.data(), p->perm.size() * 4, cudaMemcpyHostToDevice));
        p->mma.tried = false; p->mma.ok = false; p->stream.NB = 0;            // operand slabs are rebuilt from the new H on demand
    }
    p->H_dirty = false;
    return MODAL_OK;
}

// ---- vk_flow launch selection ------------------------------
int flow_capacity(size_t smem, bool ring)
{
    auto kern = ring ? md::vk_flow_kernel<true> : md::vk_flow_kernel<false>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) { cudaGetLastError(); return 0; }
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, ring ? 17 * 32 : 16 * 32, smem) != cudaSuccess) { cudaGetLastError(); return 0; }
    return per_sm;
}

// Size one team shape: schedule, residency, ring.  Returns false if it does not fit shared memory.
bool flow_shape(int nq, int nphi, int G, int force_ns, int force_res, const std::vector<uint8_t> *tile_nz, FlowConfig &c)
{
    c.G = G; c.NW = 16; c.slot_tiles = 8;
    c.sched = mh::build_flow_schedule(nq, nphi, G, c.NW, c.slot_tiles, tile_nz);
    const mh::FlowSchedule &s = c.sched;
    if (s.NLOC_MAX > 255 || s.tp_max >= (1 << 24) || s.nt > 255) return false;      // 8-bit fields of the unit descriptors
    const md::FlowSmem fixed = md::flow_smem_layout(0, c.slot_tiles, s.NQP, s.NLOC_MAX, s.U_max, s.slice_max, s.tp_max, s.stride, 0, G == 1);
    if (fixed.total + 1024 > SMEM_LIMIT) return false;
    const int avail_tiles = (int)((SMEM_LIMIT - fixed.total - 256) / 1024);
    if (force_ns <= 0 && force_res < 0 && s.tiles_max <= avail_tiles) { c.NS = 0; c.res_tiles = s.tiles_max; }
    else if (force_ns <= 0) {      // default: no ring; what is not resident is read directly from L2 by the consumers
        c.NS = 0;
        c.res_tiles = force_res >= 0 ? std::min(avail_tiles, force_res) : avail_tiles;
    } else {
        int ns = force_ns > 0 ? std::min(force_ns, 32) : std::min(20, std::max(0, (avail_tiles - 16) / c.slot_tiles));   // measured on C4: 8 -> 12 -> 16 -> 20 slots = 18.7 / 17.0 / 16.0 / 15.6 us per step
        if (ns < 2 || ns * c.slot_tiles > avail_tiles) return false;
        c.NS = ns;
        c.res_tiles = avail_tiles - ns * c.slot_tiles;
        if (force_res >= 0) c.res_tiles = std::min(c.res_tiles, force_res);
    }
    c.streamed = mh::flow_set_residency(c.sched, c.res_tiles);
    int rmax = 0;
    for (int g = 0; g < G; ++g) rmax = std::max(rmax, c.sched.blob[(size_t)g * s.stride + 6]);
    c.res_tiles = rmax;
    c.smem = md::flow_smem_layout(c.NS, c.slot_tiles, s.NQP, s.NLOC_MAX, s.U_max, s.slice_max, s.tp_max, s.stride, c.res_tiles, G == 1).total;
    return c.smem <= SMEM_LIMIT;
}

// Rough cost of one time step of one team of G CTAs while NT teams run side by side, in SM cycles.  Calibrated on
// B200 with MODAL_FLOW_TIMING: the pass over H costs ~1.5 k + 28 cycles per 1 KiB tile of a CTA; tiles
// beyond the ~187 that stay in shared memory are streamed from L2, which delivers ~3.3 KB/cycle to ALL teams together;
// the exchange phases cost 3.5 k + 70 G + 35 k / G cycles (C2: 6.3 k at G=25, 7.1 k at 50, 9.8 k at 100; C4: 15.4 k at
// 148), plus one more hop when in-plane modes are shared between CTAs.
double flow_step_cost(double tiles, int nphi, int G, int NT)
{
    const double per_cta = tiles / G;
    const double pass = 1500.0 + 28.0 * per_cta;
    const double resident_cap = 187.0;                          // tiles of shared memory
    const double streamed = std::max(0.0, per_cta - resident_cap);
    const double stream = (double)NT * G * streamed * 1024.0 / 3300.0;
    const bool shared_modes = !(G <= nphi && nphi % G == 0);
    const double exchange = G == 1 ? 0.0 : 3500.0 + 70.0 * G + 35000.0 / G + (shared_modes ? 1500.0 : 0.0);
    return std::max(pass, stream) + exchange;
}

modal_status configure_flow(modal_plan *p, int batch, FlowConfig **out)
{
    const int nq = p->d.n_q, nphi = p->d.n_phi;
    const int force_g = p->opt.flow_g, force_ns = p->opt.flow_ns, force_res = p->opt.flow_res;
    const long long key0 = ((long long)force_g << 40) | ((long long)(force_ns & 0xff) << 32) | ((long long)(force_res + 1) << 8);
    // pick the team size: minimise (rounds of samples) x (step cost) over the feasible sizes
    int bestG = 0; double best = 0;
    const int sm = p->sm_count;
    std::vector<int> cand;
    if (force_g > 0) cand.push_back(force_g);
    else {
        for (int g = 1; g <= sm; g = g < 8 ? g + 1 : g + 4) cand.push_back(g);
        cand.push_back(sm);
        for (int div = 1; div <= 4; ++div) if (nphi % div == 0 && nphi / div <= sm) cand.push_back(nphi / div);
    }
    for (int g : cand) {
        if (g < 1 || g > sm) continue;
        const double tiles_cta = (double)p->nz_tiles / g;
        if (force_g <= 0 && tiles_cta > 2000) continue;          // tables would not fit; skip the expensive build
        const int nt = std::max(1, std::min(batch, sm / g));
        const double cost = std::ceil((double)batch / nt) * flow_step_cost((double)p->nz_tiles, nphi, g, nt);
        if (!bestG || cost < best * 0.999) { bestG = g; best = cost; }
    }
    if (!bestG) { p->err += "no feasible team size for the vK flow kernel\n"; return MODAL_EINCOMPAT; }
    FlowConfig *c = nullptr;
    for (int attempt = 0; attempt < 64 && !c; ++attempt) {
        const long long key = key0 | bestG;
        FlowConfig &fc = p->flow_cfgs[key];
        if (fc.uploaded) { c = &fc; break; }
        if (flow_shape(nq, nphi, bestG, force_ns, force_res, &p->tile_nz, fc)) {
            CU(fc.dsched.ensure(fc.sched.blob.size() * 4));
            CU(cudaMemcpy(fc.dsched.p, fc.sched.blob.data(), fc.sched.blob.size() * 4, cudaMemcpyHostToDevice));
            fc.uploaded = true;
            c = &fc;
            break;
        }
        p->flow_cfgs.erase(key);
        if (force_g > 0 || bestG >= sm) break;
        bestG = std::min(sm, bestG + std::max(1, bestG / 4));    // does not fit: widen the team
    }
    if (!c) { p->err += "vK flow schedule does not fit shared memory\n"; return MODAL_EINCOMPAT; }
    const int per_sm = flow_capacity(c->smem, c->NS > 0);
    const int cap = per_sm * sm;
    if (cap < c->G) {
        char buf[128];
        snprintf(buf, sizeof buf, "a team of %d CTAs is not co-resident (capacity %d)\n", c->G, cap);
        p->err += buf;
        return MODAL_EINCOMPAT;
    }
    c->NT = std::max(1, std::min(batch, cap / c->G));
    *out = c;
    return MODAL_OK;
}

// ---- vk_mma (batched tensor-core kernel) -------------------------------------------------------
// Layout (mma_schedule.hpp), operand slabs and per-layout tables; the exchange buffers are sized per launch.
// Host part: the layout and the getters of the fp32 H values the device holds (flow tiles, internal order).
bool mma_host_layout(const modal_plan *p, mh::MmaLayout &L, const int *cluster_cap = nullptr)
{
    const int nq = p->d.n_q, nphi = p->d.n_phi;
    if (p->d.model != MODAL_VK) return false;
    // classes of the internal mode order (contiguous ranges) and of the in-plane modes: the index parities of the
    // sine-basis plate, else one class.  The K chunks a CTA multiplies come from the actual non-zeros of H.
    const bool classes = p->d.geom == MODAL_RECT && p->opt.parity_order;
    auto cls_q = [&](int k_int) { const int k = p->perm[k_int]; return classes ? (p->mq.m[k] & 1) * 2 + (p->mq.n[k] & 1) : 0; };
    std::vector<int> class_start{0};
    for (int k = 1; k < nq; ++k) if (cls_q(k) != cls_q(k - 1)) class_start.push_back(k);
    class_start.push_back(nq);
    std::vector<int> mode_class(nphi, 0);
    if (classes) for (int n = 0; n < nphi; ++n) mode_class[n] = (p->mphi.m[n] & 1) * 2 + (p->mphi.n[n] & 1);
    const std::vector<float> &Hf = p->Hf;
    const int tpn = mh::flow_tiles_per_n(nq);
    auto nz = [&](int n, int a, int b) -> bool {
        const int hi = std::max(a, b), lo = std::min(a, b), I = hi / 16, J = lo / 16;
        const size_t tile = (size_t)n * tpn + I * (I + 1) / 2 + J;
        return p->tile_nz[tile] && Hf[tile * 256 + mh::flow_elem(hi % 16, lo % 16)] != 0.f;
    };
    return mh::mma_layout(nq, nphi, p->sm_count, SMEM_LIMIT, md::mma_smem_fixed(), class_start, mode_class, nz,
                          p->opt.mma_split, p->opt.mma_ng, p->opt.mma_cluster ? cluster_cap : nullptr, L);
}

void mma_host_slabs(const modal_plan *p, const mh::MmaLayout &L, std::vector<uint16_t> &slabs)
{
    const std::vector<float> &Hf = p->Hf;
    const int tpn = mh::flow_tiles_per_n(p->d.n_q);
    auto get = [&](int n, int a, int b) -> double {
        const int hi = std::max(a, b), lo = std::min(a, b), I = hi / 16, J = lo / 16;
        const float t = Hf[((size_t)n * tpn + I * (I + 1) / 2 + J) * 256 + mh::flow_elem(hi % 16, lo % 16)];
        return hi == lo ? 2.0 * (double)t : (double)t;
    };
    mh::pack_mma_slabs(L, get, slabs);
}

modal_status configure_mma(modal_plan *p)
{
    MmaConfig &m = p->mma;
    if (m.tried) return MODAL_OK;
    m.tried = true; m.ok = false;
    // thread-block clusters of 2 / 4 / 8 CTAs of this kernel the device keeps co-resident (GPC boundaries strand some SMs)
    int ccap[9] = {0};
    if (cudaFuncSetAttribute(md::vk_mma_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_LIMIT) == cudaSuccess)
        for (int cs : {2, 4, 8}) {
            cudaLaunchConfig_t cfg{};
            cfg.gridDim = dim3(cs * 8); cfg.blockDim = dim3(md::MMA_THREADS); cfg.dynamicSmemBytes = SMEM_LIMIT;
            cudaLaunchAttribute at[1];
            at[0].id = cudaLaunchAttributeClusterDimension; at[0].val.clusterDim.x = cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
            cfg.attrs = at; cfg.numAttrs = 1;
            int n = 0;
            if (cudaOccupancyMaxActiveClusters(&n, md::vk_mma_kernel<false>, &cfg) == cudaSuccess) ccap[cs] = n;
            cudaGetLastError();
        }
    else cudaGetLastError();
    if (!mma_host_layout(p, m.L, ccap)) return MODAL_OK;
    const mh::MmaLayout &L = m.L;
    if (cudaFuncSetAttribute(md::vk_mma_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_LIMIT) != cudaSuccess) { cudaGetLastError(); return MODAL_OK; }
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, md::vk_mma_kernel<false>, md::MMA_THREADS, SMEM_LIMIT) != cudaSuccess) { cudaGetLastError(); return MODAL_OK; }
    if (per_sm * p->sm_count < L.G) return MODAL_OK;
    std::vector<uint16_t> slabs;
    mma_host_slabs(p, L, slabs);
    CU(m.dslabs.ensure(slabs.size() * 2));
    CU(cudaMemcpy(m.dslabs.p, slabs.data(), slabs.size() * 2, cudaMemcpyHostToDevice));
    std::vector<int> tab;
    auto add = [&](const std::vector<int> &v) { const size_t o = tab.size(); tab.insert(tab.end(), v.begin(), v.end()); return o; };
    m.off_nlist = add(L.nlist); m.off_klist = add(L.klist); m.off_kcnt = add(L.kcnt); m.off_fblk = add(L.fblk); m.off_fcnt = add(L.fcnt);
    std::vector<int> blk;
    for (const mh::MmaBlock &b : L.blocks) { blk.push_back(b.k0); blk.push_back(b.nb); blk.push_back(b.koff); }
    m.off_blk = add(blk);
    CU(m.dtab.ensure(tab.size() * 4));
    CU(cudaMemcpy(m.dtab.p, tab.data(), tab.size() * 4, cudaMemcpyHostToDevice));
    // owner gather: lanes per quad so that no lane has more than 16 strong loads in flight
    m.lpq = L.NGRP <= 16 ? 1 : L.NGRP <= 32 ? 2 : 4;
    m.ok = true;
    return MODAL_OK;
}

// ---- vk_stream (streaming tensor-core kernel for small / medium batches on a large tensor) -----------------
// Host part: the layout and the H stream from the fp32 H values the device holds (flow tiles, internal order).
// vk_repl: layout + device tables, once per plan and H.  Needs the parity-class structure and a symmetric H (repl_schedule.hpp); the
// grid is as many thread-block clusters as the GPU holds at once (every CTA spins on its peers: all must be resident).
modal_status configure_repl(modal_plan *p)
{
    ReplConfig &m = p->repl;
    if (m.tried) return MODAL_OK;
    m.tried = true; m.ok = false;
    if (p->d.model != MODAL_VK || p->d.n_q > md::RP_THREADS) return MODAL_OK;
    const int nq = p->d.n_q, nphi = p->d.n_phi;
    const bool classes = p->d.geom == MODAL_RECT && p->opt.parity_order;
    auto cls_q = [&](int k_int) { const int k = p->perm[k_int]; return classes ? (p->mq.m[k] & 1) * 2 + (p->mq.n[k] & 1) : 0; };
    std::vector<int> class_start{0}, cls(nq, 0);
    for (int k = 1; k < nq; ++k) if (cls_q(k) != cls_q(k - 1)) class_start.push_back(k);
    class_start.push_back(nq);
    if ((int)class_start.size() - 1 > md::RP_MAXCLS) return MODAL_OK;
    for (int c = 0; c + 1 < (int)class_start.size(); ++c) for (int k = class_start[c]; k < class_start[c + 1]; ++k) cls[k] = c;
    cudaFuncAttributes fa{};
    CU(cudaFuncGetAttributes(&fa, md::vk_repl_kernel<false>));
    cudaFuncAttributes fb{};
    CU(cudaFuncGetAttributes(&fb, md::vk_repl_kernel<true>));
    const size_t dyn_max = SMEM_LIMIT - std::max(fa.sharedSizeBytes, fb.sharedSizeBytes) - 1024;
    CU(cudaFuncSetAttribute(md::vk_repl_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn_max));
    CU(cudaFuncSetAttribute(md::vk_repl_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn_max));
    CU(cudaFuncSetAttribute(md::vk_repl_kernel<false, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn_max));
    CU(cudaFuncSetAttribute(md::vk_repl_kernel<true, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn_max));
    std::vector<double> Hi;
    const int NQ2 = (nq + 1) & ~1;
    for (int CL : {8, 4}) {
        const int SL = (((NQ2 + CL - 1) / CL) + 1) & ~1;
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(CL); cfg.blockDim = dim3(md::RP_THREADS); cfg.dynamicSmemBytes = dyn_max;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension; at[0].val.clusterDim.x = CL; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        int nc = 0;
        if (cudaOccupancyMaxActiveClusters(&nc, md::vk_repl_kernel<false>, &cfg) != cudaSuccess) { cudaGetLastError(); continue; }
        nc = std::min(nc, (nphi + CL - 1) / CL);
        if (nc < 1) continue;
        const size_t fixed = (size_t)4 + 2 * CL * SL + 16;
        if (dyn_max / 4 <= fixed) continue;
        if (Hi.empty()) { Hi.resize((size_t)nphi * nq * nq); mh::unpack_flow_tiles(nq, nphi, p->Hf, Hi.data()); }
        if (!mh::repl_layout(nq, nphi, nc * CL, dyn_max / 4 - fixed, class_start, Hi.data(), m.L)) continue;
        m.CL = CL; m.NCL = nc; m.SL = SL; m.NQ2 = NQ2;
        m.smem = md::repl_smem_bytes(m.L.hfloats_max, m.L.cp_max, m.L.rp_max, CL, SL);
        CU(m.dHp.ensure(std::max<size_t>(m.L.Hp.size(), 4) * 4));
        CU(cudaMemcpy(m.dHp.p, m.L.Hp.data(), m.L.Hp.size() * 4, cudaMemcpyHostToDevice));
        CU(m.dtab.ensure(m.L.tab.size() * 4));
        CU(cudaMemcpy(m.dtab.p, m.L.tab.data(), m.L.tab.size() * 4, cudaMemcpyHostToDevice));
        CU(m.dcls.ensure(cls.size() * 4));
        CU(cudaMemcpy(m.dcls.p, cls.data(), cls.size() * 4, cudaMemcpyHostToDevice));
        CU(m.dX.ensure((size_t)2 * nc * NQ2 * 8));
        std::vector<float>().swap(m.L.Hp);                  // the packed copy lives on the device now
        m.ok = true;
        break;
    }
    return MODAL_OK;
}

bool stream_host_layout(const modal_plan *p, int NB, mh::StreamLayout &L)
{
    if (p->d.model != MODAL_VK) return false;
    const int nq = p->d.n_q;
    const bool classes = p->d.geom == MODAL_RECT && p->opt.parity_order;
    auto cls_q = [&](int k_int) { const int k = p->perm[k_int]; return classes ? (p->mq.m[k] & 1) * 2 + (p->mq.n[k] & 1) : 0; };
    std::vector<int> class_start{0};
    for (int k = 1; k < nq; ++k) if (cls_q(k) != cls_q(k - 1)) class_start.push_back(k);
    class_start.push_back(nq);
    const std::vector<float> &Hf = p->Hf;
    const int tpn = mh::flow_tiles_per_n(nq);
    auto nz = [&](int n, int a, int b) -> bool {
        const int hi = std::max(a, b), lo = std::min(a, b), I = hi / 16, J = lo / 16;
        const size_t tile = (size_t)n * tpn + I * (I + 1) / 2 + J;
        return p->tile_nz[tile] && Hf[tile * 256 + mh::flow_elem(hi % 16, lo % 16)] != 0.f;
    };
    return mh::stream_layout(nq, p->d.n_phi, p->sm_count, NB, class_start, nz, L);
}

void stream_host_A(const modal_plan *p, const mh::StreamLayout &L, std::vector<uint16_t> &A)
{
    const std::vector<float> &Hf = p->Hf;
    const int tpn = mh::flow_tiles_per_n(p->d.n_q);
    auto get = [&](int n, int a, int b) -> double {
        const int hi = std::max(a, b), lo = std::min(a, b), I = hi / 16, J = lo / 16;
        const float t = Hf[((size_t)n * tpn + I * (I + 1) / 2 + J) * 256 + mh::flow_elem(hi % 16, lo % 16)];
        return hi == lo ? 2.0 * (double)t : (double)t;
    };
    mh::pack_stream_A(L, get, A);
}

modal_status configure_stream(modal_plan *p, int NB)
{
    StreamConfig &m = p->stream;
    if (m.NB == NB) return MODAL_OK;
    m.NB = NB; m.ok = false;
    if (!stream_host_layout(p, NB, m.L)) return MODAL_OK;
    const mh::StreamLayout &L = m.L;
    if (L.G * 4 < NB) return MODAL_OK;                   // the pickup warp of a CTA handles at most four samples
    if (md::stream_smem_layout(NB, L.rows_max, L.bch_max, L.TILE_STRIDE, 2, L.nch_max * 8192).total > SMEM_LIMIT) return MODAL_OK;
    std::vector<uint16_t> A;
    stream_host_A(p, L, A);
    CU(m.dA.ensure(A.size() * 2));
    CU(cudaMemcpy(m.dA.p, A.data(), A.size() * 2, cudaMemcpyHostToDevice));
    std::vector<int> tab;
    auto add = [&](const std::vector<int> &v) { const size_t o = tab.size(); tab.insert(tab.end(), v.begin(), v.end()); return o; };
    m.off_cta = add(L.cta_tab); m.off_tile = add(L.tile_tab);
    std::vector<int> blk;
    for (int j = 0; j < L.NKB; ++j) { blk.push_back(L.blocks[j].k0); blk.push_back(L.blocks[j].nb); blk.push_back(L.blocks[j].koff); blk.push_back(L.blk_cta0[j]); }
    m.off_blk = add(blk); m.off_nct = add(L.blk_nctas);
    CU(m.dtab.ensure(tab.size() * 4));
    CU(cudaMemcpy(m.dtab.p, tab.data(), tab.size() * 4, cudaMemcpyHostToDevice));
    // owner gather: lanes per item so that no lane has more than 12 strong loads in flight
    const int nct = *std::max_element(L.blk_nctas.begin(), L.blk_nctas.end());
    m.lpq = nct <= 12 ? 1 : nct <= 24 ? 2 : nct <= 48 ? 4 : 8;
    m.ok = true;
    return MODAL_OK;
}

template <int NB>
cudaError_t launch_stream(const md::StreamArgs &a, size_t smem, bool timing, cudaStream_t st)
{
    cudaError_t e;
    if (timing) {
        e = cudaFuncSetAttribute(md::vk_stream_kernel<NB, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        md::vk_stream_kernel<NB, true><<<a.G, md::ST_THREADS, smem, st>>>(a);
    } else {
        e = cudaFuncSetAttribute(md::vk_stream_kernel<NB, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        md::vk_stream_kernel<NB, false><<<a.G, md::ST_THREADS, smem, st>>>(a);
    }
    return cudaGetLastError();
}

template <int MPL>
cudaError_t launch_tension(const md::TensionArgs &a, cudaStream_t st)
{
    const int warps_per_block = 4;
    const int blocks = (a.batch + warps_per_block - 1) / warps_per_block;
    md::tension_kernel<MPL><<<blocks, warps_per_block * 32, 0, st>>>(a);
    return cudaGetLastError();
}

// Completes the last launch: stream synchronisation, timeout flag of the persistent kernels, first-bad steps.
modal_status finish(modal_plan *p, int *first_bad)
{
    if (!p->pending) return MODAL_OK;
    const int batch = p->last_batch;
    std::vector<int> bad(batch, -1);
    int flag = 0;
    CU(cudaSetDevice(p->device));
    CU(cudaMemcpyAsync(bad.data(), p->dbad.p, (size_t)batch * 4, cudaMemcpyDeviceToHost, p->last_stream));
    if (p->last_persistent) CU(cudaMemcpyAsync(&flag, p->dtimeout.p, 4, cudaMemcpyDeviceToHost, p->last_stream));
    CU(cudaStreamSynchronize(p->last_stream));
    p->pending = false;
    if (first_bad) memcpy(first_bad, bad.data(), (size_t)batch * 4);
    if (flag) {
        p->err += "a cross-CTA exchange of the persistent vK kernel timed out (team not co-resident?)\n";
        return MODAL_ECUDA;
    }
    for (int b = 0; b < batch; ++b)
        if (bad[b] >= 0) {
            char buf[96];
            snprintf(buf, sizeof buf, "sample %d went non-finite at step %d\n", b, bad[b]);
            p->err += buf;
            return MODAL_EUNSTABLE;
        }
    return MODAL_OK;
}

modal_status run(modal_plan *p, int batch, int n_steps, const modal_init *init, float *out_dev,
                 int *first_bad, cudaStream_t st)
{
    const modal_plan_desc &d = p->d;
    const int nq = d.n_q, P = p->NQP, cb = p->coeff_batch;
    if (p->coeffs_dirty) { modal_status s = sync_coeffs(p); if (s != MODAL_OK) return s; }
    if (p->H_dirty) { modal_status s = sync_H(p); if (s != MODAL_OK) return s; }
    CU(cudaSetDevice(p->device));
    // initial state, masked and padded:  v^0 = q^0 - q^-1
    std::vector<double> q0((size_t)batch * P, 0.0), v0((size_t)batch * P, 0.0), gain;
    for (int b = 0; b < batch; ++b)
        for (int k = 0; k < nq; ++k) {
            if (!p->active[(size_t)(cb == 1 ? 0 : b) * nq + k]) continue;
            const double q = init->q0[(size_t)b * nq + k];
            q0[(size_t)b * P + p->iperm[k]] = q;
            if (init->qm1) v0[(size_t)b * P + p->iperm[k]] = q - init->qm1[(size_t)b * nq + k];
        }
    CU(p->dq0.ensure(q0.size() * 8)); CU(p->dv0.ensure(v0.size() * 8)); CU(p->dbad.ensure((size_t)batch * 4));
    CU(cudaMemcpyAsync(p->dq0.p, q0.data(), q0.size() * 8, cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(p->dv0.p, v0.data(), v0.size() * 8, cudaMemcpyHostToDevice, st));
    if (init->fext_signal) {
        gain.assign((size_t)batch * P, 0.0);
        for (int b = 0; b < batch; ++b)
            for (int k = 0; k < nq; ++k)
                if (p->active[(size_t)(cb == 1 ? 0 : b) * nq + k]) gain[(size_t)b * P + p->iperm[k]] = init->fext_gain[(size_t)b * nq + k];
        CU(p->dgain.ensure(gain.size() * 8));
        CU(cudaMemcpyAsync(p->dgain.p, gain.data(), gain.size() * 8, cudaMemcpyHostToDevice, st));
    }
    CU(cudaMemsetAsync(p->dbad.p, 0xff, (size_t)batch * 4, st));
    CU(p->dtimeout.ensure(4));
    CU(cudaMemsetAsync(p->dtimeout.p, 0, 4, st));
    bool persistent = false;
    const int auto_start = init->qm1 ? 0 : 1;
    const double half_T2 = 0.5 * p->T * p->T;

    // vK kernel family: the batched tensor-core kernel when H fits the shared memory of the GPU (batch >= 64), the streaming
    // tensor-core kernel when it does not (batch >= 8), else the FP32 flow kernel; "vk_impl" forces one
    bool use_mma = false, use_stream = false;
    // small systems (the paper's 10-mode benchmark point): one warp per sample, no barriers, no exchange (vk_small.cuh)
    const bool use_small = d.model == MODAL_VK && nq <= 32 && d.n_phi <= 32 && (long long)d.n_phi * nq * nq <= 8192 &&
                           (p->opt.vk_impl == 0 || p->opt.vk_impl == 4) && p->opt.flow_g == 0 && p->opt.flow_ns == 0 && p->opt.flow_res < 0;
    if (d.model == MODAL_VK && p->opt.vk_impl == 4 && !use_small) { p->err += "vk_impl=4: the small-system kernel needs N_q, N_phi <= 32 and N_phi N_q^2 <= 8192\n"; return MODAL_EINCOMPAT; }
    // mid-size systems at small batch: a team of CTAs per sample with replicated state and one hop per step (vk_dense.cuh), when
    // the dense H of a CTA's modes fits shared memory
    bool use_dense = false;
    int dn_G = 0, dn_per_launch = 0, dn_ld = (nq + 3) & ~3;
    size_t dn_smem = 0;
    if (d.model == MODAL_VK && !use_small && nq <= md::DN_THREADS && (p->opt.vk_impl == 5 || (p->opt.vk_impl == 0 && batch < 64)) &&
        p->opt.flow_g == 0 && p->opt.flow_ns == 0 && p->opt.flow_res < 0) {
        dn_per_launch = std::min(batch, p->sm_count);
        dn_G = std::min({p->sm_count / dn_per_launch, d.n_phi, md::DN_G_MAX, 8 * std::min(md::DN_THREADS / dn_ld, 8)});
        const int modes_max = (d.n_phi + dn_G - 1) / dn_G;
        dn_smem = (size_t)modes_max * nq * dn_ld * 4;
        use_dense = dn_G >= 2 && dn_smem + 16 * 1024 <= SMEM_LIMIT;
        // batches of 8 and more have the streaming tensor-core kernel as alternative: keep the team kernel only while a CTA has few modes
        if (p->opt.vk_impl == 0 && batch >= 8 && modes_max > 8) use_dense = false;
        if (p->opt.vk_impl == 5 && !use_dense) { p->err += "vk_impl=5: the dense H of a CTA's modes does not fit shared memory (or one CTA per sample)\n"; return MODAL_EINCOMPAT; }
    }
    // one sample of a plate too large for the team kernel: replicated state, whole in-plane modes per CTA, one hop per step (vk_repl.cuh)
    bool use_repl = false;
    if (d.model == MODAL_VK && !use_small && !use_dense && (p->opt.vk_impl == 6 || (p->opt.vk_impl == 0 && batch == 1)) &&
        p->opt.flow_g == 0 && p->opt.flow_ns == 0 && p->opt.flow_res < 0) {
        if (batch == 1) { modal_status s = configure_repl(p); if (s != MODAL_OK) return s; use_repl = p->repl.ok; }
        if (p->opt.vk_impl == 6 && !use_repl) { p->err += "vk_impl=6: the replicated-state kernel takes one sample of a plan whose H has the parity-class structure and fits shared memory\n"; return MODAL_EINCOMPAT; }
    }
    if (d.model == MODAL_VK && !use_small && !use_dense && !use_repl) {
        const int impl = p->opt.vk_impl;
        if ((impl == 0 && batch >= 64) || impl == 2) { modal_status s = configure_mma(p); if (s != MODAL_OK) return s; use_mma = p->mma.ok; }
        if (!use_mma && ((impl == 0 && batch >= 8) || impl == 3)) {
            const int NB = batch <= 16 ? 16 : batch <= 32 ? 32 : 64;
            modal_status s = configure_stream(p, NB); if (s != MODAL_OK) return s;
            use_stream = p->stream.ok;
            if (impl == 3 && !use_stream) { p->err += "vk_impl=3: the streaming kernel has no layout for this plan\n"; return MODAL_EINCOMPAT; }
        }
    }
    if (d.model != MODAL_VK) {
        md::TensionArgs a{};
        a.batch = batch; a.n_steps = n_steps; a.n_modes_pad = P; a.coeff_stride = cb == 1 ? 0 : P;
        a.kv = p->dkv.as<double>(); a.kq = p->dkq.as<double>(); a.r = p->dr.as<double>(); a.astart = p->dast.as<double>();
        a.lambda = p->dlam.as<float>(); a.w = p->dw.as<float>(); a.c = p->dc.as<float>();
        a.q0 = p->dq0.as<double>(); a.v0 = p->dv0.as<double>();
        a.auto_start = auto_start; a.half_T2 = half_T2;
        a.fext = init->fext_signal; a.gain = p->dgain.as<double>();
        a.out = out_dev; a.traj = init->traj_dev; a.n_q = nq; a.first_bad = p->dbad.as<int>();
        cudaError_t e;
        switch (P / 32) {
            case 1: e = launch_tension<1>(a, st); break;
            case 2: e = launch_tension<2>(a, st); break;
            case 3: e = launch_tension<3>(a, st); break;
            case 4: e = launch_tension<4>(a, st); break;
            case 5: e = launch_tension<5>(a, st); break;
            case 6: e = launch_tension<6>(a, st); break;
            case 7: e = launch_tension<7>(a, st); break;
            case 8: e = launch_tension<8>(a, st); break;
            case 9: e = launch_tension<9>(a, st); break;
            case 10: e = launch_tension<10>(a, st); break;
            case 11: e = launch_tension<11>(a, st); break;
            case 12: e = launch_tension<12>(a, st); break;
            case 13: e = launch_tension<13>(a, st); break;
            case 14: e = launch_tension<14>(a, st); break;
            case 15: e = launch_tension<15>(a, st); break;
            case 16: e = launch_tension<16>(a, st); break;
            default: p->err += "n_q too large for the tension kernel of this build (n_q <= 512)\n"; return MODAL_EINCOMPAT;
        }
        CU(e);
        p->kinfo[0] = 1; p->kinfo[1] = 1; p->kinfo[2] = (batch + 3) / 4; p->kinfo[3] = 128;
        p->kinfo[4] = 0; p->kinfo[5] = 1; p->kinfo[6] = 0; p->kinfo[7] = P;
    } else if (use_small) {
        if (!p->small_H_valid) {
            const size_t nH = (size_t)d.n_phi * nq * nq;
            std::vector<double> Hi(nH);
            mh::unpack_flow_tiles(nq, d.n_phi, p->Hf, Hi.data());
            std::vector<float> Hd(nH);
            for (size_t i = 0; i < nH; ++i) Hd[i] = (float)Hi[i];
            CU(p->dHsmall.ensure(nH * 4));
            CU(cudaMemcpy(p->dHsmall.p, Hd.data(), nH * 4, cudaMemcpyHostToDevice));
            p->small_H_valid = true;
        }
        md::SmallArgs a{};
        a.Hd = p->dHsmall.as<float>(); a.n_q = nq; a.n_phi = d.n_phi; a.NQP = P; a.batch = batch; a.n_steps = n_steps;
        a.coeff_stride_q = cb == 1 ? 0 : P; a.coeff_stride_phi = cb == 1 ? 0 : d.n_phi;
        a.kv = p->dkv.as<double>(); a.kq = p->dkq.as<double>(); a.r = p->dr.as<double>(); a.astart = p->dast.as<double>();
        a.s = p->ds.as<float>(); a.w = p->dw.as<float>();
        a.q0 = p->dq0.as<double>(); a.v0 = p->dv0.as<double>();
        a.auto_start = auto_start; a.half_T2 = half_T2;
        a.fext = init->fext_signal; a.gain = p->dgain.as<double>();
        a.out = out_dev; a.traj = init->traj_dev; a.kperm = p->dperm.as<int>(); a.first_bad = p->dbad.as<int>();
        const size_t smem = md::small_smem_bytes(nq, d.n_phi);
        const bool hreg = nq <= 16 && d.n_phi * nq <= 128;
        CU(cudaFuncSetAttribute(md::vk_small_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        CU(cudaFuncSetAttribute(md::vk_small_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        const int blocks = (batch + md::SM_WARPS - 1) / md::SM_WARPS;
        if (hreg) md::vk_small_kernel<true><<<blocks, md::SM_WARPS * 32, smem, st>>>(a);
        else md::vk_small_kernel<false><<<blocks, md::SM_WARPS * 32, smem, st>>>(a);
        CU(cudaGetLastError());
        p->kinfo[0] = 2; p->kinfo[1] = 1; p->kinfo[2] = blocks; p->kinfo[3] = md::SM_WARPS * 32;
        p->kinfo[4] = (int)smem; p->kinfo[5] = 1; p->kinfo[6] = 0; p->kinfo[7] = P;
    } else if (use_dense) {
        if (!p->dense_H_valid) {
            const size_t nH = (size_t)d.n_phi * nq * nq;
            std::vector<double> Hi(nH);
            mh::unpack_flow_tiles(nq, d.n_phi, p->Hf, Hi.data());
            std::vector<float> Hd((size_t)d.n_phi * nq * dn_ld, 0.f);
            for (int n = 0; n < d.n_phi; ++n)
                for (int a_ = 0; a_ < nq; ++a_)
                    for (int b_ = 0; b_ < nq; ++b_) Hd[((size_t)n * nq + a_) * dn_ld + b_] = (float)Hi[((size_t)n * nq + a_) * nq + b_];
            CU(p->dHdense.ensure(Hd.size() * 4));
            CU(cudaMemcpy(p->dHdense.p, Hd.data(), Hd.size() * 4, cudaMemcpyHostToDevice));
            p->dense_H_valid = true;
        }
        const size_t nscr = (size_t)2 * dn_per_launch * dn_G * nq * 8;
        CU(p->ddscr.ensure(nscr));
        CU(cudaFuncSetAttribute(md::vk_dense_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dn_smem));
        int out_cta = 0, fewest = 1 << 30;                     // the pickup goes to a CTA with the fewest modes
        for (int g = 0; g < dn_G; ++g) {
            const int cnt = (int)((long long)d.n_phi * (g + 1) / dn_G) - (int)((long long)d.n_phi * g / dn_G);
            if (cnt < fewest) { fewest = cnt; out_cta = g; }
        }
        for (int b0 = 0; b0 < batch; b0 += dn_per_launch) {
            const int nb = std::min(dn_per_launch, batch - b0);
            md::DenseArgs a{};
            a.n_q = nq; a.n_phi = d.n_phi; a.NQP = P; a.batch = nb; a.n_steps = n_steps; a.G = dn_G; a.ld = dn_ld;
            a.NJ = std::max(1, std::min(md::DN_THREADS / (dn_ld / 4), nq)); a.out_cta = out_cta;
            a.coeff_stride_q = cb == 1 ? 0 : 1; a.coeff_stride_phi = cb == 1 ? 0 : 1;
            const size_t oq = cb == 1 ? 0 : (size_t)b0 * P, op = cb == 1 ? 0 : (size_t)b0 * d.n_phi;
            a.H = p->dHdense.as<float>();
            a.kv = p->dkv.as<double>() + oq; a.kq = p->dkq.as<double>() + oq; a.r = p->dr.as<double>() + oq; a.astart = p->dast.as<double>() + oq;
            a.s = p->ds.as<float>() + op; a.w = p->dw.as<float>() + oq;
            a.q0 = p->dq0.as<double>() + (size_t)b0 * P; a.v0 = p->dv0.as<double>() + (size_t)b0 * P;
            a.auto_start = auto_start; a.half_T2 = half_T2;
            a.fext = init->fext_signal ? init->fext_signal + (size_t)b0 * n_steps : nullptr;
            a.gain = init->fext_signal ? p->dgain.as<double>() + (size_t)b0 * P : nullptr;
            a.out = out_dev + (size_t)b0 * n_steps;
            a.traj = init->traj_dev ? init->traj_dev + (size_t)b0 * n_steps * nq : nullptr; a.kperm = p->dperm.as<int>();
            a.first_bad = p->dbad.as<int>() + b0;
            a.scratch = p->ddscr.as<unsigned long long>(); a.timeout_flag = p->dtimeout.as<int>();
            CU(cudaMemsetAsync(p->ddscr.p, 0, (size_t)2 * nb * dn_G * nq * 8, st));
            md::vk_dense_kernel<<<nb * dn_G, md::DN_THREADS, dn_smem, st>>>(a);
            CU(cudaGetLastError());
        }
        persistent = true;
        p->kinfo[0] = 6; p->kinfo[1] = dn_G; p->kinfo[2] = dn_per_launch; p->kinfo[3] = md::DN_THREADS;
        p->kinfo[4] = (int)dn_smem; p->kinfo[5] = 1 | 2; p->kinfo[6] = 0; p->kinfo[7] = P;
    } else if (use_repl) {
        ReplConfig &m = p->repl;
        md::ReplArgs a{};
        a.n_q = nq; a.NQ2 = m.NQ2; a.n_phi = d.n_phi; a.NQP = P; a.n_steps = n_steps; a.G = m.L.G; a.CL = m.CL; a.NCL = m.NCL; a.SL = m.SL;
        a.out_cta = m.L.out_cta; a.hfloats_max = m.L.hfloats_max; a.cp_max = m.L.cp_max; a.rp_max = m.L.rp_max;
        a.Hp = m.dHp.as<float>(); a.tab = m.dtab.as<int>(); a.cls = m.dcls.as<int>();
        a.kv = p->dkv.as<double>(); a.kq = p->dkq.as<double>(); a.r = p->dr.as<double>(); a.astart = p->dast.as<double>();
        a.s = p->ds.as<float>(); a.w = p->dw.as<float>();
        a.q0 = p->dq0.as<double>(); a.v0 = p->dv0.as<double>();
        a.auto_start = auto_start; a.half_T2 = half_T2;
        a.fext = init->fext_signal; a.gain = init->fext_signal ? p->dgain.as<double>() : nullptr;
        a.out = out_dev; a.traj = init->traj_dev; a.kperm = p->dperm.as<int>(); a.first_bad = p->dbad.as<int>();
        a.X = m.dX.as<unsigned long long>(); a.timeout_flag = p->dtimeout.as<int>();
        CU(cudaMemsetAsync(m.dX.p, 0, (size_t)2 * m.NCL * m.NQ2 * 8, st));
        const bool timing = p->opt.timing != 0;
        if (timing) {
            CU(p->dtiming.ensure((size_t)m.L.G * 64));
            CU(cudaMemsetAsync(p->dtiming.p, 0, (size_t)m.L.G * 64, st));
            a.timing = p->dtiming.as<long long>();
        }
        {
            cudaLaunchConfig_t cfg{};
            cfg.gridDim = dim3(m.L.G); cfg.blockDim = dim3(md::RP_THREADS); cfg.dynamicSmemBytes = m.smem; cfg.stream = st;
            cudaLaunchAttribute at[1];
            at[0].id = cudaLaunchAttributeClusterDimension; at[0].val.clusterDim.x = m.CL; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
            cfg.attrs = at; cfg.numAttrs = 1;
            int mm = 0;
            for (int nm : m.L.cta_nmodes) mm = std::max(mm, nm);
            if (timing && mm <= 2) CU(cudaLaunchKernelEx(&cfg, md::vk_repl_kernel<true, 2>, a));
            else if (timing) CU(cudaLaunchKernelEx(&cfg, md::vk_repl_kernel<true, md::RP_MAXM>, a));
            else if (mm <= 2) CU(cudaLaunchKernelEx(&cfg, md::vk_repl_kernel<false, 2>, a));
            else CU(cudaLaunchKernelEx(&cfg, md::vk_repl_kernel<false, md::RP_MAXM>, a));
        }
        CU(cudaGetLastError());
        if (timing) {
            CU(cudaStreamSynchronize(st));
            std::vector<long long> tm((size_t)m.L.G * 8);
            CU(cudaMemcpy(tm.data(), p->dtiming.p, tm.size() * 8, cudaMemcpyDeviceToHost));
            double acc[8] = {0}, mx[8] = {0};
            for (size_t x = 0; x < tm.size(); ++x) { acc[x & 7] += (double)tm[x]; mx[x & 7] = std::max(mx[x & 7], (double)tm[x]); }
            const double den = (double)m.L.G * n_steps;
            fprintf(stderr, "[modal repl timing] G=%d clusters of %d, H <= %d KiB per CTA, rows per item <= %d  cycles/step mean | max over CTAs:\n"
                            "   items (partials of t = H q) %.0f | %.0f   join + block sums %.0f | %.0f   cluster reduce-scatter + publish %.0f | %.0f   gather %.0f | %.0f\n",
                    m.L.G, m.CL, m.L.hfloats_max / 256, m.L.rows_max, acc[0] / den, mx[0] / n_steps, acc[1] / den, mx[1] / n_steps,
                    acc[2] / den, mx[2] / n_steps, acc[3] / den, mx[3] / n_steps);
        }
        persistent = true;
        p->kinfo[0] = 8; p->kinfo[1] = m.L.G; p->kinfo[2] = m.CL; p->kinfo[3] = md::RP_THREADS;
        p->kinfo[4] = (int)m.smem; p->kinfo[5] = 1 | 2; p->kinfo[6] = m.L.rows_max; p->kinfo[7] = P;
    } else if (use_stream) {
        StreamConfig &m = p->stream;
        const mh::StreamLayout &L = m.L;
        const int NB = m.NB;
        const int stage_bytes = L.nch_max * 8192;                  // one tile per ring stage
        const size_t base = md::stream_smem_layout(NB, L.rows_max, L.bch_max, L.TILE_STRIDE, 0, stage_bytes).total;
        int nstg = (int)std::min<size_t>(md::ST_NSTG_MAX, (SMEM_LIMIT - base) / stage_bytes);
        if (p->opt.mma_nstg > 0) nstg = std::min(nstg, std::max(p->opt.mma_nstg, 2));
        if (nstg < 2) { p->err += "streaming vK kernel: no room for the operand ring\n"; return MODAL_EINCOMPAT; }
        const size_t smem = md::stream_smem_layout(NB, L.rows_max, L.bch_max, L.TILE_STRIDE, nstg, stage_bytes).total;
        const int KOP = L.KC * 16;
        const size_t nqx = (size_t)NB * KOP * 4, nGx = (size_t)d.n_phi * L.NKB * NB * 4, nfx = (size_t)L.G * 128 * NB * 4, npx = (size_t)4 * L.G * NB * 16 + 256;
        CU(m.dqx.ensure(nqx)); CU(m.dGx.ensure(nGx)); CU(m.dfx.ensure(nfx)); CU(m.dpx.ensure(npx));
        const bool timing = p->opt.timing != 0;
        for (int b0 = 0; b0 < batch; b0 += NB) {
            const int nb = std::min(NB, batch - b0);
            md::StreamArgs a{};
            const int *tab = m.dtab.as<int>();
            a.A = m.dA.as<uint16_t>(); a.cta_tab = tab + m.off_cta; a.tile_tab = tab + m.off_tile; a.tile_stride = L.TILE_STRIDE;
            a.blk = tab + m.off_blk; a.blk_nctas = tab + m.off_nct;
            a.NKB = L.NKB; a.KOP = KOP; a.G = L.G; a.NSTG = nstg; a.stage_bytes = stage_bytes; a.rows_max = L.rows_max; a.bch_max = L.bch_max; a.LPQ = m.lpq;
            a.n_q = nq; a.n_phi = d.n_phi; a.NQP = P; a.batch = nb; a.n_steps = n_steps;
            a.coeff_stride_q = cb == 1 ? 0 : P; a.coeff_stride_phi = cb == 1 ? 0 : d.n_phi;
            const size_t oq = cb == 1 ? 0 : (size_t)b0 * P;
            a.kv = p->dkv.as<double>() + oq; a.kq = p->dkq.as<double>() + oq; a.r = p->dr.as<double>() + oq; a.astart = p->dast.as<double>() + oq;
            a.s = p->ds.as<float>() + (cb == 1 ? 0 : (size_t)b0 * d.n_phi); a.w = p->dw.as<float>() + oq;
            a.q0 = p->dq0.as<double>() + (size_t)b0 * P; a.v0 = p->dv0.as<double>() + (size_t)b0 * P;
            a.auto_start = auto_start; a.half_T2 = half_T2;
            a.fext = init->fext_signal ? init->fext_signal + (size_t)b0 * n_steps : nullptr;
            a.gain = init->fext_signal ? p->dgain.as<double>() + (size_t)b0 * P : nullptr;
            a.out = out_dev + (size_t)b0 * n_steps;
            a.traj = init->traj_dev ? init->traj_dev + (size_t)b0 * n_steps * nq : nullptr; a.kperm = p->dperm.as<int>();
            a.first_bad = p->dbad.as<int>() + b0;
            // exchange buffers (L2 resident); everything starts at tag / epoch 0 (the first step uses 1)
            CU(cudaMemsetAsync(m.dqx.p, 0, nqx, st)); CU(cudaMemsetAsync(m.dGx.p, 0, nGx, st));
            CU(cudaMemsetAsync(m.dfx.p, 0, nfx, st)); CU(cudaMemsetAsync(m.dpx.p, 0, npx, st));
            a.qx = m.dqx.as<uint32_t>(); a.Gx = m.dGx.as<uint32_t>(); a.fx = m.dfx.as<uint32_t>(); a.px = m.dpx.as<unsigned long long>();
            a.wflag = reinterpret_cast<uint32_t *>(m.dpx.as<unsigned char>() + (size_t)4 * L.G * NB * 16);
            a.timeout_flag = p->dtimeout.as<int>();
            if (timing) {
                CU(p->dtiming.ensure((size_t)L.G * 128));
                CU(cudaMemsetAsync(p->dtiming.p, 0, (size_t)L.G * 128, st));
                a.timing = p->dtiming.as<long long>();
            }
            persistent = true;
            CU(NB == 16 ? launch_stream<16>(a, smem, timing, st) : NB == 32 ? launch_stream<32>(a, smem, timing, st) : launch_stream<64>(a, smem, timing, st));
            if (timing) {
                CU(cudaStreamSynchronize(st));
                std::vector<long long> tm((size_t)L.G * 16);
                CU(cudaMemcpy(tm.data(), p->dtiming.p, tm.size() * 8, cudaMemcpyDeviceToHost));
                double acc[16] = {0};
                for (size_t x = 0; x < tm.size(); ++x) acc[x & 15] += (double)tm[x];
                const double den = (double)L.G * n_steps;
                double mx[16] = {0}; int amx[16] = {0};
                for (size_t x = 0; x < tm.size(); ++x) if ((double)tm[x] > mx[x & 15]) { mx[x & 15] = (double)tm[x]; amx[x & 15] = (int)(x >> 4); }
                static const char *names[16] = {"E q operand (wait + build)", "E own rows", "E wait acc", "E epi1 (all tiles, incl. wait)", "E G wait (sentinels)", "E epi2 (incl. G wait)",
                                                "E f store", "E q seen (sentinels) after", "O gather", "O update + publish", "O barrier + pickup", "O wait for own E", "M step's MMAs", "M waiting for H chunks", "own f stored -> forces gathered", ""};
                fprintf(stderr, "[modal stream timing] G=%d NB=%d blocks=%d tiles/CTA<=%d chunks/CTA<=%d rows/CTA<=%d ring=%d lpq=%d  cycles/step: mean over CTAs | max (CTA)\n",
                        L.G, NB, L.NKB, L.tiles_max, L.bch_max, L.rows_max, nstg, m.lpq);
                for (int x = 0; x < 16; ++x)
                    if (names[x][0]) fprintf(stderr, "   %-32s %8.0f | %8.0f (%d: %d tiles, block %d)\n", names[x], acc[x] / den, mx[x] / n_steps, amx[x], L.cta_ntiles[amx[x]], L.cta_block[amx[x]]);
            }
        }
        p->kinfo[0] = 5; p->kinfo[1] = L.G; p->kinfo[2] = NB; p->kinfo[3] = md::ST_THREADS;
        p->kinfo[4] = (int)smem; p->kinfo[5] = 1 | 2; p->kinfo[6] = L.tiles_max; p->kinfo[7] = P;
    } else if (use_mma) {
        MmaConfig &m = p->mma;
        const mh::MmaLayout &L = m.L;
        // M tiles per launch: as many (<= 8) as leave room for one tile's worth of ring stages beside slab and owner state; a wider batch
        // runs as consecutive launches of equal size
        int mt_cap = md::MMA_MT_MAX;
        while (mt_cap > 1 && md::mma_smem_layout((int)L.slab_bytes, mt_cap, L.rows_max, L.RBQ, std::max(2, L.KCL)).total > SMEM_LIMIT) --mt_cap;
        const int tiles = (batch + 127) / 128, launches = (tiles + mt_cap - 1) / mt_cap;
        const int chunk = 128 * ((tiles + launches - 1) / launches);
        size_t smem = 0;
        for (int b0 = 0; b0 < batch; b0 += chunk) {
            const int nb = std::min(chunk, batch - b0), MT = (nb + 127) / 128;
            const size_t base = md::mma_smem_layout((int)L.slab_bytes, MT, L.rows_max, L.RBQ, 0).total;
            int nstg = base < SMEM_LIMIT ? (int)std::min<size_t>(md::MMA_NSTG_MAX, (SMEM_LIMIT - base) / 8192) : 0;
            if (p->opt.mma_nstg > 0) nstg = std::min(nstg, p->opt.mma_nstg);
            if (nstg < 2) { p->err += "batched vK kernel: no room for the operand ring\n"; return MODAL_EINCOMPAT; }
            smem = md::mma_smem_layout((int)L.slab_bytes, MT, L.rows_max, L.RBQ, nstg).total;
            CU(cudaFuncSetAttribute(md::vk_mma_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            CU(cudaFuncSetAttribute(md::vk_mma_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            md::MmaArgs a{};
            a.slabs = m.dslabs.as<uint16_t>(); a.slab_bytes = (int)L.slab_bytes; a.NSTG = nstg;
            a.NKB = L.NKB; a.NGRP = L.NGRP; a.NG = L.NG; a.NG4 = L.NG4; a.NC = L.NC; a.S = L.S; a.RBT = L.RBT; a.RBQ = L.RBQ;
            a.KC = L.KC; a.KCL = L.KCL; a.G = L.G; a.rows_max = L.rows_max; a.LPQ = m.lpq; a.CL = L.CL;
            const int *tab = m.dtab.as<int>();
            a.nlist = tab + m.off_nlist; a.klist = tab + m.off_klist; a.kcnt = tab + m.off_kcnt; a.fblk = tab + m.off_fblk;
            a.fcnt = tab + m.off_fcnt; a.blk = tab + m.off_blk;
            a.n_q = nq; a.n_phi = d.n_phi; a.NQP = P;
            a.batch = nb; a.n_steps = n_steps; a.MT = MT;
            a.coeff_stride_q = cb == 1 ? 0 : P; a.coeff_stride_phi = cb == 1 ? 0 : d.n_phi;
            const size_t oq = cb == 1 ? 0 : (size_t)b0 * P;
            a.kv = p->dkv.as<double>() + oq; a.kq = p->dkq.as<double>() + oq; a.r = p->dr.as<double>() + oq;
            a.astart = p->dast.as<double>() + oq; a.sT = p->dsT.as<float>() + (cb == 1 ? 0 : b0); a.sT_stride = cb; a.w = p->dw.as<float>() + oq;
            a.q0 = p->dq0.as<double>() + (size_t)b0 * P; a.v0 = p->dv0.as<double>() + (size_t)b0 * P;
            a.auto_start = auto_start; a.half_T2 = half_T2;
            a.fext = init->fext_signal ? init->fext_signal + (size_t)b0 * n_steps : nullptr;
            a.gain = init->fext_signal ? p->dgain.as<double>() + (size_t)b0 * P : nullptr;
            a.out = out_dev + (size_t)b0 * n_steps;
            a.traj = init->traj_dev ? init->traj_dev + (size_t)b0 * n_steps * nq : nullptr; a.kperm = p->dperm.as<int>();
            a.first_bad = p->dbad.as<int>() + b0;
            // exchange buffers (L2 resident); everything starts at tag / epoch 0 (the first step uses 1)
            const size_t nQop = (size_t)MT * L.KC * 8192, nqf = (size_t)MT * L.NKB * L.RBQ * 128 * 16,
                         nGx = (size_t)2 * MT * L.NGRP * L.NKB * 128 * 16 * L.NG4, nfx = (size_t)MT * L.NGRP * L.NKB * L.RBQ * 128 * 16,
                         nfl = (size_t)MT * L.NKB * L.NGRP * md::MMA_FS * 4, npx = (size_t)2 * MT * L.NKB * 128 * 16;
            CU(m.dQop.ensure(nQop)); CU(m.dqf.ensure(nqf)); CU(m.dGx.ensure(nGx)); CU(m.dfx.ensure(nfx)); CU(m.dflags.ensure(nfl)); CU(m.dpx.ensure(npx));
            CU(cudaMemsetAsync(m.dQop.p, 0, nQop, st)); CU(cudaMemsetAsync(m.dqf.p, 0, nqf, st)); CU(cudaMemsetAsync(m.dGx.p, 0, nGx, st));
            CU(cudaMemsetAsync(m.dfx.p, 0, nfx, st)); CU(cudaMemsetAsync(m.dflags.p, 0, nfl, st)); CU(cudaMemsetAsync(m.dpx.p, 0, npx, st));
            a.Qop = m.dQop.as<uint16_t>(); a.qf = m.dqf.as<float>(); a.Gx = m.dGx.as<uint32_t>(); a.fx = m.dfx.as<uint32_t>();
            a.qflag = m.dflags.as<unsigned>(); a.px = m.dpx.as<unsigned long long>();
            a.timeout_flag = p->dtimeout.as<int>();
            const bool timing = p->opt.timing != 0;
            if (timing) {
                CU(p->dtiming.ensure((size_t)L.G * (128 + 256)));
                CU(cudaMemsetAsync(p->dtiming.p, 0, (size_t)L.G * (128 + 256), st));
                a.timing = p->dtiming.as<long long>();
                a.trace = a.timing + (size_t)L.G * 16;
            }
            persistent = true;
            {
                cudaLaunchConfig_t cfg{};
                cfg.gridDim = dim3(L.G); cfg.blockDim = dim3(md::MMA_THREADS); cfg.dynamicSmemBytes = smem; cfg.stream = st;
                cudaLaunchAttribute at[1];
                at[0].id = cudaLaunchAttributeClusterDimension; at[0].val.clusterDim.x = L.CL ? L.NKB : 1; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
                cfg.attrs = at; cfg.numAttrs = 1;
                CU(timing ? cudaLaunchKernelEx(&cfg, md::vk_mma_kernel<true>, a) : cudaLaunchKernelEx(&cfg, md::vk_mma_kernel<false>, a));
            }
            CU(cudaGetLastError());
            if (timing) {
                CU(cudaStreamSynchronize(st));
                std::vector<long long> tm((size_t)L.G * 16);
                CU(cudaMemcpy(tm.data(), p->dtiming.p, tm.size() * 8, cudaMemcpyDeviceToHost));
                double acc[16] = {0};
                for (size_t x = 0; x < tm.size(); ++x) acc[x & 15] += (double)tm[x];
                const double den = (double)L.G * n_steps;
                fprintf(stderr, "[modal mma timing] G=%d (%d groups x %d blocks%s) NG=%d NC=%d S=%d KCL=%d ring=%d MT=%d  cycles/step of tile 0, mean over CTAs:\n"
                        "   E: wait q %.0f | wait acc %.0f | epi1+send %.0f (first unit in registers after %.0f, all units after %.0f) | G hop %.0f | epi2 %.0f\n"
                        "   O: gather %.0f | update %.0f | publish %.0f | barrier+fence+flag %.0f     P: flag poll %.0f   M: first chunk -> commit %.0f\n"
                        "   hops: end of epilogue 2 -> forces gathered %.0f | own flag set -> all source flags seen %.0f\n",
                        L.G, L.NGRP, L.NKB, L.CL ? ", clusters" : "", L.NG, L.NC, L.S, L.KCL, nstg, MT, acc[0] / den, acc[1] / den, acc[2] / den, acc[5] / den, acc[6] / den, acc[3] / den, acc[4] / den,
                        acc[8] / den, acc[11] / den, acc[9] / den, acc[10] / den, acc[12] / den, acc[13] / den, acc[14] / den, acc[15] / den);
                if (n_steps >= 68) {   // spread of the phase boundaries of step 65 over the CTAs (globaltimer, ns after the earliest event of the step)
                    std::vector<long long> tr((size_t)L.G * 32);
                    CU(cudaMemcpy(tr.data(), p->dtiming.as<long long>() + (size_t)L.G * 16, tr.size() * 8, cudaMemcpyDeviceToHost));
                    static const char *names[8] = {"q ready (flags seen)", "accumulator ready", "G sent", "G received", "epilogue 2 done", "forces gathered",
                                                   "q published", "flag released"};
                    long long t0 = -1;
                    for (int c = 0; c < L.G; ++c) for (int e = 0; e < 8; ++e) { const long long v = tr[((size_t)c * 4 + 1) * 8 + e]; if (v > 0 && (t0 < 0 || v < t0)) t0 = v; }
                    for (int e = 0; e < 8; ++e) {
                        std::vector<long long> v;
                        for (int c = 0; c < L.G; ++c) if (tr[((size_t)c * 4 + 1) * 8 + e] > 0) v.push_back(tr[((size_t)c * 4 + 1) * 8 + e] - t0);
                        if (v.empty()) continue;
                        std::sort(v.begin(), v.end());
                        fprintf(stderr, "   step 65 %-20s ns after the step's first event: min %6lld  p10 %6lld  median %6lld  p90 %6lld  max %6lld\n", names[e], v.front(),
                                v[v.size() / 10], v[v.size() / 2], v[v.size() * 9 / 10], v.back());
                    }
                }
            }
        }
        p->kinfo[0] = 4; p->kinfo[1] = L.G; p->kinfo[2] = L.NGRP; p->kinfo[3] = md::MMA_THREADS;
        p->kinfo[4] = (int)smem; p->kinfo[5] = 1 | 2; p->kinfo[6] = L.S; p->kinfo[7] = P;
    } else {
        FlowConfig *c = nullptr;
        modal_status s = configure_flow(p, batch, &c);
        if (s != MODAL_OK) return s;
        const mh::FlowSchedule &fs = c->sched;
        md::FlowArgs a{};
        a.Hf = p->dHf.as<float>(); a.sched = c->dsched.as<int>(); a.sched_stride = fs.stride;
        a.off_units = fs.off_units; a.off_ltile = fs.off_ltile; a.off_pieces = fs.off_pieces; a.off_pu = fs.off_pu;
        a.off_kbptr = fs.off_kbptr; a.off_kblist = fs.off_kblist;
        a.G = c->G; a.NT = c->NT; a.NW = c->NW; a.NS = c->NS; a.slot_tiles = c->slot_tiles; a.direct = c->NS == 0 ? 1 : 0;
        a.NQP = P; a.n_q = nq; a.n_phi = d.n_phi; a.nb = fs.nb;
        a.U_max = fs.U_max; a.tp_max = fs.tp_max; a.NLOC_MAX = fs.NLOC_MAX; a.res_tiles = c->res_tiles;
        a.slice_max = fs.slice_max; a.MS = fs.MS;
        a.batch = batch; a.n_steps = n_steps;
        a.coeff_stride_q = cb == 1 ? 0 : P; a.coeff_stride_phi = cb == 1 ? 0 : d.n_phi;
        a.kv = p->dkv.as<double>(); a.kq = p->dkq.as<double>(); a.r = p->dr.as<double>(); a.astart = p->dast.as<double>();
        a.s = p->ds.as<float>(); a.w = p->dw.as<float>();
        a.q0 = p->dq0.as<double>(); a.v0 = p->dv0.as<double>();
        a.auto_start = auto_start; a.half_T2 = half_T2;
        a.fext = init->fext_signal; a.gain = p->dgain.as<double>();
        a.out = out_dev; a.traj = init->traj_dev; a.kperm = p->dperm.as<int>(); a.first_bad = p->dbad.as<int>();
        if ((long long)((batch + c->NT - 1) / c->NT) * n_steps >= 0xffffffffLL) { p->err += "batch x n_steps too large for one launch\n"; return MODAL_EINCOMPAT; }
        if (c->G > 1) {
            const size_t nfx = (size_t)c->NT * c->G * P * 8, ngx = (size_t)c->NT * d.n_phi * fs.MS * 8, nqx = (size_t)c->NT * md::FLOW_QREP * P * 8;
            CU(p->dfx.ensure(nfx)); CU(p->dgx.ensure(ngx)); CU(p->dqx.ensure(nqx));
            CU(cudaMemsetAsync(p->dfx.p, 0, nfx, st)); CU(cudaMemsetAsync(p->dgx.p, 0, ngx, st)); CU(cudaMemsetAsync(p->dqx.p, 0, nqx, st));
            a.fx = p->dfx.as<unsigned long long>(); a.gx = p->dgx.as<unsigned long long>(); a.qx = p->dqx.as<unsigned long long>();
        }
        a.timeout_flag = p->dtimeout.as<int>();
        const bool timing = p->opt.timing != 0;
        if (timing) {
            CU(p->dtiming.ensure((size_t)c->G * c->NT * 64));
            CU(cudaMemsetAsync(p->dtiming.p, 0, (size_t)c->G * c->NT * 64, st));
            a.timing = p->dtiming.as<long long>();
        }
        persistent = true;
        if (c->NS > 0) {
            CU(cudaFuncSetAttribute(md::vk_flow_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem));
            md::vk_flow_kernel<true><<<c->G * c->NT, (c->NW + 1) * 32, c->smem, st>>>(a);
        } else {
            CU(cudaFuncSetAttribute(md::vk_flow_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem));
            md::vk_flow_kernel<false><<<c->G * c->NT, c->NW * 32, c->smem, st>>>(a);
        }
        CU(cudaGetLastError());
        if (timing) {   // diagnostics: mean cycles per time step and phase over the CTAs
            CU(cudaStreamSynchronize(st));
            std::vector<long long> tm((size_t)c->G * c->NT * 8);
            CU(cudaMemcpy(tm.data(), p->dtiming.p, tm.size() * 8, cudaMemcpyDeviceToHost));
            double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0}, mx0 = 0;
            for (size_t i = 0; i < tm.size(); ++i) { acc[i & 7] += (double)tm[i]; if ((i & 7) == 0) mx0 = std::max(mx0, (double)tm[i]); }
            const double den = (double)c->G * c->NT * n_steps * ((batch + c->NT - 1) / c->NT);
            fprintf(stderr, "[modal flow timing] G=%d NT=%d NS=%d res=%d cycles/step: A %.0f (max %.0f)  B1 %.0f  B2 %.0f  C %.0f  D+barrier %.0f  total %.0f\n",
                    c->G, c->NT, c->NS, c->res_tiles, acc[0] / den, mx0 * c->G * c->NT / den, acc[1] / den, acc[4] / den, acc[5] / den, acc[6] / den, acc[3] / den);
        }
        p->kinfo[0] = 3; p->kinfo[1] = c->G; p->kinfo[2] = c->NT; p->kinfo[3] = (c->NW + (c->NS > 0 ? 1 : 0)) * 32;
        p->kinfo[4] = (int)c->smem; p->kinfo[5] = (c->streamed == 0 ? 1 : 0) | (c->G > 1 ? 2 : 0); p->kinfo[6] = c->NS; p->kinfo[7] = P;
    }
    p->last_stream = st; p->last_batch = batch; p->last_persistent = persistent; p->pending = true;
    return first_bad ? finish(p, first_bad) : MODAL_OK;
}

modal_status check_sim_args(modal_plan *p, int batch, int n_steps, const modal_init *init, const void *out)
{
    if (!p) return MODAL_EINVAL;
    p->err.clear();
    if (p->device < 0) { p->err = "plan has no CUDA device (host-only plan): there is no CPU fallback\n"; return MODAL_ECUDA; }
    if (batch < 1 || batch > p->d.max_batch) p->err += "batch outside [1, max_batch]\n";
    if (n_steps < 1 || n_steps > p->d.max_steps) p->err += "n_steps outside [1, max_steps]\n";
    if (!init || !init->q0) p->err += "init->q0 is required\n";
    if (init && init->fext_signal && !init->fext_gain) p->err += "fext_signal needs fext_gain\n";
    if (!out) p->err += "output buffer is NULL\n";
    if (p->coeff_batch != 1 && p->coeff_batch != batch) p->err += "coeff_batch must be 1 or equal to batch\n";
    return p->err.empty() ? MODAL_OK : MODAL_EINVAL;
}

}  // namespace

// ============================================================================ C ABI ====

extern "C" modal_status modal_plan_create(const modal_plan_desc *desc, int cuda_device, modal_plan **out)
{
    if (out) *out = nullptr;
    g_create_error.clear();
    if (!desc || !out) { g_create_error = "desc and out must not be NULL\n"; return MODAL_EINVAL; }
    if (!validate_desc(*desc, g_create_error)) return MODAL_EINVAL;
    modal_plan *p = new (std::nothrow) modal_plan;
    if (!p) return MODAL_ENOMEM;
    p->d = *desc; p->device = cuda_device; p->T = 1.0 / desc->sample_rate;
    const modal_plan_desc &d = p->d;
    const int nq = d.n_q;
    if (d.geom == MODAL_RECT) {
        p->mq = mh::rect_modes(d.Lx, d.Ly, nq);
        if (d.model == MODAL_VK) p->mphi = mh::rect_modes(d.Lx, d.Ly, d.n_phi);   // reading R5
    } else p->mq = mh::string_modes(d.Lx, nq);
    p->NQP = d.model == MODAL_VK ? mh::flow_padded_nq(nq) : ((nq + 31) / 32) * 32;
    build_perm(p);
    p->coeff_batch = 1;
    p->omega.resize(nq); p->sigma.resize(nq); p->pickup.resize(nq); p->lambda_s.resize(nq);
    p->nl_scale.resize(n_nl(p));
    modal_sample_geom g = fill_geom(p, nullptr);
    derive_row(p, g, p->omega.data(), p->sigma.data(), p->nl_scale.data(), p->lambda_s.data(), p->pickup.data());
    if (d.model == MODAL_VK) {
        const double geom = mh::H_geom(d.Lx, d.Ly);
        const mh::ModeSet &q = p->mq, &f = p->mphi;
        auto get = [&](int n, int a, int b) {
            return geom * mh::H_bracket(q.m[a], q.n[a], q.m[b], q.n[b], f.m[n], f.n[n]);
        };
        set_H(p, get);
        p->zeta4.resize(d.n_phi);
        for (int n = 0; n < d.n_phi; ++n) p->zeta4[n] = p->mphi.lambda[n] * p->mphi.lambda[n];      // reading R5
    }
    if (cuda_device >= 0) {
        cudaError_t e = cudaSetDevice(cuda_device);
        cudaDeviceProp prop{};
        if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, cuda_device);
        if (e != cudaSuccess) {
            g_create_error = std::string("CUDA error: ") + cudaGetErrorString(e) + "\n";
            delete p;
            return MODAL_ECUDA;
        }
        if (prop.major != 10) {
            g_create_error = "this library is built for sm_100a (B200) only\n";
            delete p;
            return MODAL_ECUDA;
        }
        p->sm_count = prop.multiProcessorCount;
    }
    modal_status s = sync_coeffs(p);
    if (s == MODAL_OK) s = sync_H(p);
    if (s != MODAL_OK) { g_create_error = p->err; modal_plan_destroy(p); return s; }
    *out = p;
    return MODAL_OK;
}

extern "C" modal_status modal_coeffs_upload(modal_plan *p, const modal_coeffs *c)
{
    if (!p || !c) return MODAL_EINVAL;
    p->err.clear();
    const modal_plan_desc &d = p->d;
    const int nq = d.n_q, nnl = n_nl(p), cb = c->coeff_batch;
    if (cb < 1 || cb > d.max_batch) { p->err = "coeff_batch outside [1, max_batch]\n"; return MODAL_EINVAL; }
    if (c->H_full && d.model != MODAL_VK) { p->err = "H_full given but the plan is not MODAL_VK\n"; return MODAL_EINVAL; }
    if (c->lambda && d.model == MODAL_VK) { p->err = "lambda is a MODAL_TENSION / MODAL_LINEAR coefficient\n"; return MODAL_EINVAL; }
    auto finite = [&](const double *a, size_t n, const char *name) {
        for (size_t i = 0; a && i < n; ++i)
            if (!std::isfinite(a[i])) { p->err += std::string(name) + " contains non-finite values\n"; return; }
    };
    finite(c->omega, (size_t)cb * nq, "omega"); finite(c->sigma, (size_t)cb * nq, "sigma");
    finite(c->nl_scale, (size_t)cb * nnl, "nl_scale"); finite(c->lambda, (size_t)cb * nq, "lambda");
    finite(c->pickup, (size_t)cb * nq, "pickup"); finite(c->H_full, c->H_full ? (size_t)d.n_phi * nq * nq : 0, "H_full");
    for (size_t i = 0; c->omega && i < (size_t)cb * nq; ++i) if (c->omega[i] < 0) { p->err += "omega must be non-negative\n"; break; }
    for (size_t i = 0; c->sigma && i < (size_t)cb * nq; ++i) if (c->sigma[i] < 0) { p->err += "sigma must be non-negative\n"; break; }
    if (c->H_full) {
        double mx = 0, asym = 0;
        for (size_t i = 0; i < (size_t)d.n_phi * nq * nq; ++i) mx = std::max(mx, std::fabs(c->H_full[i]));
        for (int n = 0; n < d.n_phi; ++n)
            for (int a = 0; a < nq; ++a)
                for (int b = 0; b < a; ++b)
                    asym = std::max(asym, std::fabs(c->H_full[((size_t)n * nq + a) * nq + b] - c->H_full[((size_t)n * nq + b) * nq + a]));
        if (asym > 1e-12 * mx) p->err += "H_full is not symmetric in its two transverse indices\n";
    }
    if (!p->err.empty()) return MODAL_EINVAL;
    // re-shape the per-sample arrays to the new coeff_batch (row 0 broadcast when it changes)
    auto reshape = [&](std::vector<double> &v, int width, const double *src) {
        if (src) { v.assign(src, src + (size_t)cb * width); return; }
        if (cb == p->coeff_batch) return;
        std::vector<double> row(v.begin(), v.begin() + width), nv((size_t)cb * width);
        for (int b = 0; b < cb; ++b) std::copy(row.begin(), row.end(), nv.begin() + (size_t)b * width);
        v.swap(nv);
    };
    reshape(p->omega, nq, c->omega); reshape(p->sigma, nq, c->sigma); reshape(p->nl_scale, nnl, c->nl_scale);
    reshape(p->lambda_s, nq, c->lambda); reshape(p->pickup, nq, c->pickup);
    p->coeff_batch = cb;
    p->coeffs_dirty = true;
    if (c->H_full) {
        const double *H = c->H_full;
        auto get = [&](int n, int a, int b) { return H[((size_t)n * nq + a) * nq + b]; };
        set_H(p, get);
    }
    modal_status s = sync_coeffs(p);
    if (s == MODAL_OK && p->H_dirty) s = sync_H(p);
    return s;
}

extern "C" modal_status modal_simulate(modal_plan *p, int batch, int n_steps, const modal_init *init,
                                       float *out_audio_dev, int *first_bad_step, void *cuda_stream)
{
    modal_status s = check_sim_args(p, batch, n_steps, init, out_audio_dev);
    if (s != MODAL_OK) return s;
    return run(p, batch, n_steps, init, out_audio_dev, first_bad_step, (cudaStream_t)cuda_stream);
}

extern "C" modal_status modal_simulate_host(modal_plan *p, int batch, int n_steps, const modal_init *init,
                                            float *out_audio_host, int *first_bad_step)
{
    modal_status s = check_sim_args(p, batch, n_steps, init, out_audio_host);
    if (s != MODAL_OK) return s;
    const size_t bytes = (size_t)batch * n_steps * 4;
    CU(cudaSetDevice(p->device));
    CU(p->dout.ensure(bytes));
    if (p->pinned_bytes < bytes) {                       // pinned staging: the D2H copy runs at PCIe speed
        if (p->pinned_out) cudaFreeHost(p->pinned_out);
        p->pinned_out = nullptr; p->pinned_bytes = 0;
        CU(cudaMallocHost(&p->pinned_out, bytes));
        p->pinned_bytes = bytes;
    }
    s = run(p, batch, n_steps, init, p->dout.as<float>(), nullptr, nullptr);
    if (s != MODAL_OK) return s;
    CU(cudaMemcpyAsync(p->pinned_out, p->dout.p, bytes, cudaMemcpyDeviceToHost, nullptr));
    std::vector<int> bad(batch, -1);
    s = finish(p, bad.data());
    if (s != MODAL_OK && s != MODAL_EUNSTABLE) return s;
    memcpy(out_audio_host, p->pinned_out, bytes);
    if (first_bad_step) memcpy(first_bad_step, bad.data(), (size_t)batch * 4);
    return s;
}

// ---- reverse pass (vk_bptt.cuh) ---------------------------------------------------------------------
namespace {
// d(c1, c2, c3)/d(omega, sigma) of q+ = c1 q + c2 q- - c3 f:  SV PAPER.md:163-167 Eq. 21-23;  FTM PAPER.md:147-151 Eq. 16-18 (R7)
struct CoeffDerivs { double c1_w, c1_g, c2_g, c3_w, c3_g; };
CoeffDerivs coeff_derivs(int scheme, double w, double g, double T)
{
    CoeffDerivs d{};
    if (scheme == MODAL_SV) {
        const double den = 1.0 + g * T;
        d.c1_w = -2.0 * w * T * T / den; d.c1_g = -(2.0 - w * w * T * T) * T / (den * den);
        d.c2_g = 2.0 * T / (den * den);
        d.c3_w = 0.0; d.c3_g = -T * T * T / (den * den);
    } else {
        const double wt = std::sqrt(w * w - g * g), e = std::exp(-g * T), sn = std::sin(wt * T), cs = std::cos(wt * T);
        const double wt_w = w / wt, wt_g = -g / wt;
        const double dc3 = T * e * (T * cs * wt - sn) / (wt * wt);
        d.c1_w = -2.0 * e * sn * T * wt_w; d.c1_g = -2.0 * T * e * cs - 2.0 * e * sn * T * wt_g;
        d.c2_g = 2.0 * T * std::exp(-2.0 * g * T);
        d.c3_w = dc3 * wt_w; d.c3_g = -T * T * e * sn / wt + dc3 * wt_g;
    }
    return d;
}
}  // namespace

extern "C" modal_status modal_bptt(modal_plan *p, int batch, int n_steps, const modal_bptt_args *ar, void *cuda_stream)
{
    if (!p) return MODAL_EINVAL;
    p->err.clear();
    const modal_plan_desc &d = p->d;
    const bool vk = d.model == MODAL_VK;
    const int nq = d.n_q, nphi = vk ? d.n_phi : 1, cb = p->coeff_batch;      // tension / linear: one non-linear scale per sample
    if (p->device < 0) { p->err += "modal_bptt needs a CUDA device: there is no CPU fallback\n"; return MODAL_ECUDA; }
    if (!ar || batch < 1 || n_steps < 1 || batch > d.max_batch || n_steps > d.max_steps || (cb != 1 && cb != batch)) {
        p->err += "modal_bptt: batch / n_steps outside the plan, or coeff_batch neither 1 nor batch\n"; return MODAL_EINVAL;
    }
    if (!ar->qm1 || !ar->traj_dev || !ar->gout_dev) { p->err += "modal_bptt: qm1, traj_dev and gout_dev are required\n"; return MODAL_EINVAL; }
    if (nq > md::BP_THREADS_MAX) { p->err += "modal_bptt: n_q <= 512 in this build\n"; return MODAL_EINCOMPAT; }
    if (p->pending) { modal_status s = finish(p, nullptr); if (s != MODAL_OK && s != MODAL_EUNSTABLE) return s; }
    CU(cudaSetDevice(p->device));
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    enum { B_H, B_C1, B_C2, B_C3, B_S, B_W, B_QM1, B_GQ0, B_GQM1, B_GC1, B_GC2, B_GC3, B_GW, B_GS, B_AUX, B_SCR };
    // dense fp32 H in plan order (once per H)
    const size_t nH = (size_t)nphi * nq * nq;
    const int ld = (nq + 3) & ~3;                                   // row stride: 16-byte loads
    if (vk && !p->bp_H_valid) {
        std::vector<double> Hi(nH);
        mh::unpack_flow_tiles(nq, nphi, p->Hf, Hi.data());
        std::vector<float> Hu((size_t)nphi * nq * ld, 0.f);
        for (int n = 0; n < nphi; ++n)
            for (int a = 0; a < nq; ++a)
                for (int b = 0; b < nq; ++b) Hu[((size_t)n * nq + p->perm[a]) * ld + p->perm[b]] = (float)Hi[((size_t)n * nq + a) * nq + b];
        CU(p->bp[B_H].ensure(Hu.size() * 4));
        CU(cudaMemcpy(p->bp[B_H].p, Hu.data(), Hu.size() * 4, cudaMemcpyHostToDevice));
        p->bp_H_valid = true;
    }
    // canonical coefficients in plan order (masked modes: zero rows, as in the forward kernels)
    std::vector<double> c1((size_t)cb * nq, 0.0), c2(c1), c3(c1);
    std::vector<float> w((size_t)cb * nq, 0.f), s((size_t)cb * nphi);
    std::vector<int> act((size_t)cb * nq, 0);
    for (int b = 0; b < cb; ++b)
        for (int k = 0; k < nq; ++k) {
            const size_t o = (size_t)b * nq + k;
            const double om = p->omega[o], sg = p->sigma[o];
            if (!(mh::mode_active(d.scheme, om, sg, p->T) && std::isfinite(om) && std::isfinite(sg))) continue;
            if (d.scheme == MODAL_FTM && !(om > sg)) { p->err += "modal_bptt: FTM scheme with an overdamped mode\n"; return MODAL_EINVAL; }
            const mh::StepCoeffs c = mh::step_coeffs(d.scheme, om, sg, p->T);
            act[o] = 1; c1[o] = 1.0 + c.kv - c.kq; c2[o] = -c.kv; c3[o] = c.r; w[o] = (float)p->pickup[o];
        }
    for (size_t i = 0; i < s.size(); ++i) s[i] = (float)p->nl_scale[i];
    std::vector<double> qm1((size_t)batch * nq);
    for (int b = 0; b < batch; ++b)
        for (int k = 0; k < nq; ++k) qm1[(size_t)b * nq + k] = act[(size_t)(cb == 1 ? 0 : b) * nq + k] ? ar->qm1[(size_t)b * nq + k] : 0.0;
    auto up = [&](int i, const void *src, size_t bytes) -> cudaError_t {
        cudaError_t e = p->bp[i].ensure(bytes);
        return e != cudaSuccess ? e : cudaMemcpyAsync(p->bp[i].p, src, bytes, cudaMemcpyHostToDevice, st);
    };
    CU(up(B_C1, c1.data(), c1.size() * 8)); CU(up(B_C2, c2.data(), c2.size() * 8)); CU(up(B_C3, c3.data(), c3.size() * 8));
    CU(up(B_S, s.data(), s.size() * 4)); CU(up(B_W, w.data(), w.size() * 4)); CU(up(B_QM1, qm1.data(), qm1.size() * 8));
    const size_t nbq = (size_t)batch * nq * 8, nbs = (size_t)batch * nphi * 8;
    for (int i : {B_GQ0, B_GQM1, B_GC1, B_GC2, B_GC3, B_GW}) CU(p->bp[i].ensure(nbq));
    CU(p->bp[B_GS].ensure(nbs));
    CU(cudaMemsetAsync(p->bp[B_GS].p, 0, nbs, st));
    const bool wantH = vk && ar->grad_H != nullptr;
    const size_t n_mu = (size_t)batch * n_steps * nq * 4, n_sc = (size_t)batch * n_steps * nphi * 4;
    if (wantH) CU(p->bp[B_AUX].ensure(n_mu + 2 * n_sc + nH * 8));
    CU(p->dtimeout.ensure(4));
    CU(cudaMemsetAsync(p->dtimeout.p, 0, 4, st));
    if (!vk) {
        // tension-modulated / linear models: one warp per sample (tension_bptt_kernel); lambda travels in the dense-H buffer slot
        std::vector<float> lam((size_t)cb * nq, 0.f);
        if (d.model == MODAL_TENSION) for (size_t i = 0; i < lam.size(); ++i) lam[i] = act[i] ? (float)p->lambda_s[i] : 0.f;
        if (d.model != MODAL_TENSION) for (float &x : s) x = 0.f;
        CU(up(B_H, lam.data(), lam.size() * 4)); CU(up(B_S, s.data(), s.size() * 4));
        md::TensionBpttArgs a{};
        a.n_q = nq; a.batch = batch; a.n_steps = n_steps; a.cb_q = cb == 1 ? 0 : nq;
        a.c1 = p->bp[B_C1].as<double>(); a.c2 = p->bp[B_C2].as<double>(); a.c3 = p->bp[B_C3].as<double>();
        a.w = p->bp[B_W].as<float>(); a.lam = p->bp[B_H].as<float>(); a.c = p->bp[B_S].as<float>();
        a.traj = ar->traj_dev; a.qm1 = p->bp[B_QM1].as<double>(); a.gout = ar->gout_dev;
        a.g_q0 = p->bp[B_GQ0].as<double>(); a.g_qm1 = p->bp[B_GQM1].as<double>(); a.g_c1 = p->bp[B_GC1].as<double>();
        a.g_c2 = p->bp[B_GC2].as<double>(); a.g_c3 = p->bp[B_GC3].as<double>(); a.g_w = p->bp[B_GW].as<double>(); a.g_c = p->bp[B_GS].as<double>();
        const size_t smem = md::tension_bptt_smem(nq);
        CU(cudaFuncSetAttribute(md::tension_bptt_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        md::tension_bptt_kernel<<<(batch + md::TB_WARPS - 1) / md::TB_WARPS, md::TB_WARPS * 32, smem, st>>>(a);
        CU(cudaGetLastError());
    }
    // launches of co-resident teams: G CTAs per sample, samples per launch <= SMs
    const int per_launch = std::min(batch, p->sm_count);
    int G = std::min({p->sm_count / per_launch, nphi, md::BP_G_MAX, 8 * std::min(md::BP_THREADS_MAX / ((nq + 3) & ~3), 8)});
    const size_t nscr = (size_t)2 * per_launch * G * nq * 16;
    CU(p->bp[B_SCR].ensure(std::max<size_t>(nscr, 16)));
    const int threads = md::BP_THREADS_MAX;
    // the modes of a CTA stay in shared memory when they fit (C2: 4 modes x 40 KB); otherwise H streams from L2 every step
    const int modes_max = (nphi + G - 1) / G;
    const size_t hs_bytes = (size_t)modes_max * nq * ld * 4;
    const int resident = hs_bytes + 28 * 1024 <= SMEM_LIMIT ? 1 : 0;
    const int NJ = std::max(1, std::min(md::BP_THREADS_MAX / (ld / 4), nq));
    const size_t dyn = resident ? hs_bytes : 0;
    if (resident) CU(cudaFuncSetAttribute(md::vk_bptt_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
    for (int b0 = 0; vk && b0 < batch; b0 += per_launch) {
        const int nb = std::min(per_launch, batch - b0);
        md::BpttArgs a{};
        a.n_q = nq; a.n_phi = nphi; a.batch = nb; a.n_steps = n_steps; a.G = G; a.ld = ld; a.NJ = NJ;
        a.cb_q = cb == 1 ? 0 : nq; a.cb_phi = cb == 1 ? 0 : nphi;
        const size_t oq = cb == 1 ? 0 : (size_t)b0 * nq, op = cb == 1 ? 0 : (size_t)b0 * nphi;
        a.H = p->bp[B_H].as<float>();
        a.c1 = p->bp[B_C1].as<double>() + oq; a.c2 = p->bp[B_C2].as<double>() + oq; a.c3 = p->bp[B_C3].as<double>() + oq;
        a.s = p->bp[B_S].as<float>() + op; a.w = p->bp[B_W].as<float>() + oq;
        a.traj = ar->traj_dev + (size_t)b0 * n_steps * nq; a.qm1 = p->bp[B_QM1].as<double>() + (size_t)b0 * nq;
        a.gout = ar->gout_dev + (size_t)b0 * n_steps;
        const size_t ob = (size_t)b0 * nq;
        a.g_q0 = p->bp[B_GQ0].as<double>() + ob; a.g_qm1 = p->bp[B_GQM1].as<double>() + ob; a.g_c1 = p->bp[B_GC1].as<double>() + ob;
        a.g_c2 = p->bp[B_GC2].as<double>() + ob; a.g_c3 = p->bp[B_GC3].as<double>() + ob; a.g_w = p->bp[B_GW].as<double>() + ob;
        a.g_s = p->bp[B_GS].as<double>() + (size_t)b0 * nphi;
        if (wantH) {
            unsigned char *aux = p->bp[B_AUX].as<unsigned char>();
            a.mu_traj = reinterpret_cast<float *>(aux) + (size_t)b0 * n_steps * nq;
            a.dsc = reinterpret_cast<float *>(aux + n_mu) + (size_t)b0 * n_steps * nphi;
            a.esc = reinterpret_cast<float *>(aux + n_mu + n_sc) + (size_t)b0 * n_steps * nphi;
        }
        a.scratch = p->bp[B_SCR].as<unsigned long long>();
        a.timeout_flag = p->dtimeout.as<int>();
        if (G > 1) CU(cudaMemsetAsync(p->bp[B_SCR].p, 0, (size_t)2 * nb * G * nq * 16, st));
        if (resident) md::vk_bptt_kernel<true><<<nb * G, threads, dyn, st>>>(a);
        else md::vk_bptt_kernel<false><<<nb * G, threads, 0, st>>>(a);
        CU(cudaGetLastError());
    }
    std::vector<double> gH;
    if (wantH) {
        unsigned char *aux = p->bp[B_AUX].as<unsigned char>();
        double *dgH = reinterpret_cast<double *>(aux + n_mu + 2 * n_sc);
        md::vk_gradH_kernel<<<dim3(nphi, (nq + 15) / 16), threads, 0, st>>>(nq, nphi, batch, n_steps, ar->traj_dev, reinterpret_cast<const float *>(aux),
                                                                          reinterpret_cast<const float *>(aux + n_mu), reinterpret_cast<const float *>(aux + n_mu + n_sc), dgH);
        CU(cudaGetLastError());
        CU(cudaMemcpyAsync(ar->grad_H, dgH, nH * 8, cudaMemcpyDeviceToHost, st));
    }
    std::vector<double> gc1((size_t)batch * nq), gc2(gc1), gc3(gc1);
    int flag = 0;
    auto down = [&](int i, double *dst, size_t bytes) -> cudaError_t { return dst ? cudaMemcpyAsync(dst, p->bp[i].p, bytes, cudaMemcpyDeviceToHost, st) : cudaSuccess; };
    CU(down(B_GQ0, ar->grad_q0, nbq)); CU(down(B_GQM1, ar->grad_qm1, nbq)); CU(down(B_GW, ar->grad_pickup, nbq)); CU(down(B_GS, ar->grad_nl_scale, nbs));
    CU(down(B_GC1, gc1.data(), nbq)); CU(down(B_GC2, gc2.data(), nbq)); CU(down(B_GC3, gc3.data(), nbq));
    CU(cudaMemcpyAsync(&flag, p->dtimeout.p, 4, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    if (flag) { p->err += "modal_bptt: a cross-CTA exchange timed out (team not co-resident?)\n"; return MODAL_ECUDA; }
    // the forward recurrence uses -c3 f: dL/dc3 as defined in modal.h (q+ = c1 q + c2 q- + c3 (fext - f)) is what the kernel accumulated
    for (int b = 0; b < batch; ++b)
        for (int k = 0; k < nq; ++k) {
            const size_t o = (size_t)b * nq + k, oc = (size_t)(cb == 1 ? 0 : b) * nq + k;
            if (ar->grad_c1) ar->grad_c1[o] = gc1[o];
            if (ar->grad_c2) ar->grad_c2[o] = gc2[o];
            if (ar->grad_c3) ar->grad_c3[o] = gc3[o];
            double gw_ = 0.0, gg_ = 0.0;
            if (act[oc]) {
                const CoeffDerivs cd = coeff_derivs(d.scheme, p->omega[oc], p->sigma[oc], p->T);
                gw_ = gc1[o] * cd.c1_w + gc3[o] * cd.c3_w;
                gg_ = gc1[o] * cd.c1_g + gc2[o] * cd.c2_g + gc3[o] * cd.c3_g;
            }
            if (ar->grad_omega) ar->grad_omega[o] = gw_;
            if (ar->grad_sigma) ar->grad_sigma[o] = gg_;
        }
    return MODAL_OK;
}

extern "C" modal_status modal_plan_check(modal_plan *p, int *first_bad_step)
{
    if (!p) return MODAL_EINVAL;
    if (p->device < 0) { p->err = "plan has no CUDA device (host-only plan)\n"; return MODAL_ECUDA; }
    return finish(p, first_bad_step);
}

extern "C" modal_status modal_plan_set_option(modal_plan *p, const char *key, int value)
{
    if (!p || !key) return MODAL_EINVAL;
    p->err.clear();
    struct { const char *name; int *field; int lo, hi; } tab[] = {
        {"vk_impl", &p->opt.vk_impl, 0, 6}, {"flow_g", &p->opt.flow_g, 0, 1024}, {"flow_ns", &p->opt.flow_ns, 0, 32},
        {"flow_res", &p->opt.flow_res, -1, 1 << 20}, {"mma_split", &p->opt.mma_split, 0, 4}, {"mma_ng", &p->opt.mma_ng, 0, 8},
        {"mma_nstg", &p->opt.mma_nstg, 0, 16}, {"mma_cluster", &p->opt.mma_cluster, 0, 1}, {"parity_order", &p->opt.parity_order, 0, 1}, {"timing", &p->opt.timing, 0, 1}};
    for (auto &t : tab)
        if (!strcmp(key, t.name)) {
            if (value < t.lo || value > t.hi) { p->err = std::string("option ") + key + ": value out of range\n"; return MODAL_EINVAL; }
            if (*t.field == value) return MODAL_OK;
            const int old = *t.field;
            *t.field = value;
            if (t.field == &p->opt.parity_order && p->d.model == MODAL_VK) {
                // re-pack H in the new internal order (user-order copy through the old permutation)
                const int nq = p->d.n_q, nphi = p->d.n_phi;
                std::vector<double> Hi((size_t)nphi * nq * nq), Hu((size_t)nphi * nq * nq);
                mh::unpack_flow_tiles(nq, nphi, p->Hf, Hi.data());
                for (int n = 0; n < nphi; ++n)
                    for (int a = 0; a < nq; ++a)
                        for (int b = 0; b < nq; ++b)
                            Hu[((size_t)n * nq + p->perm[a]) * nq + p->perm[b]] = Hi[((size_t)n * nq + a) * nq + b];
                (void)old;
                build_perm(p);
                set_H(p, [&](int n, int a, int b) { return Hu[((size_t)n * nq + a) * nq + b]; });
                p->coeffs_dirty = true;
            }
            if (t.field == &p->opt.mma_split || t.field == &p->opt.mma_ng || t.field == &p->opt.mma_cluster) { p->mma.tried = false; p->mma.ok = false; }
            if (t.field == &p->opt.parity_order) p->stream.NB = 0;
            return MODAL_OK;
        }
    p->err = std::string("unknown option ") + key + "\n";
    return MODAL_EINVAL;
}

extern "C" modal_status modal_plan_set_airy_basis(modal_plan *p, int basis, int n_trial)
{
    if (!p) return MODAL_EINVAL;
    p->err.clear();
    const modal_plan_desc &d = p->d;
    if (d.model != MODAL_VK) { p->err = "the in-plane basis belongs to MODAL_VK plans\n"; return MODAL_EINVAL; }
    if ((basis != MODAL_AIRY_SINE && basis != MODAL_AIRY_CLAMPED_RITZ) || n_trial < 0 || n_trial > 64) {
        p->err = "basis must be MODAL_AIRY_SINE or MODAL_AIRY_CLAMPED_RITZ, n_trial in [0, 64]\n"; return MODAL_EINVAL;
    }
    const int nphi = d.n_phi;
    const mh::ModeSet &q = p->mq;
    if (basis == MODAL_AIRY_SINE) {
        const double geom = mh::H_geom(d.Lx, d.Ly);
        const mh::ModeSet &f = p->mphi;
        set_H(p, [&](int n, int a, int b) { return geom * mh::H_bracket(q.m[a], q.n[a], q.m[b], q.n[b], f.m[n], f.n[n]); });
        for (int n = 0; n < nphi; ++n) p->zeta4[n] = f.lambda[n] * f.lambda[n];
    } else {
        // trial functions per axis: enough for the n_phi lowest modes with a margin (the highest kept mode has ~sqrt(n_phi) half-waves per axis)
        int nt = n_trial > 0 ? n_trial : std::max(12, 2 * (int)std::ceil(std::sqrt(1.5 * nphi * std::max(d.Lx / d.Ly, d.Ly / d.Lx))) + 6);
        nt = std::min(nt, 64);
        mh::AiryRitz R;
        if (nt * nt < nphi || !mh::airy_ritz_basis(d.Lx, d.Ly, nphi, nt, R)) {
            p->err = "Rayleigh-Ritz Airy basis: too few trial functions for n_phi, or the mass matrix is not positive definite\n";
            return MODAL_EINCOMPAT;
        }
        set_H(p, [&](int n, int a, int b) {
            return mh::airy_ritz_H_entry(nt, &R.c[(size_t)n * nt * nt], d.Lx, d.Ly, q.m[a], q.n[a], q.m[b], q.n[b]);
        });
        p->zeta4 = R.zeta4;
    }
    p->airy_basis = basis;
    for (int b = 0; b < p->coeff_batch; ++b)
        for (int n = 0; n < nphi; ++n) p->nl_scale[(size_t)b * nphi + n] = d.E / (2.0 * d.rho * p->zeta4[n]);
    p->coeffs_dirty = true;
    modal_status s = sync_coeffs(p);
    if (s == MODAL_OK && p->H_dirty) s = sync_H(p);
    return s;
}

extern "C" void modal_plan_destroy(modal_plan *p)
{
    if (!p) return;
    if (p->device >= 0) {
        cudaSetDevice(p->device);
        if (p->pending) cudaStreamSynchronize(p->last_stream);
        for (DevBuf *b : {&p->dkv, &p->dkq, &p->dr, &p->dast, &p->ds, &p->dsT, &p->dw, &p->dlam, &p->dc, &p->dq0, &p->dv0, &p->dgain, &p->dbad,
                          &p->dout, &p->dHf, &p->dfx, &p->dgx, &p->dqx, &p->dtiming, &p->dperm, &p->dtimeout, &p->mma.dslabs, &p->mma.dtab,
                          &p->mma.dQop, &p->mma.dqf, &p->mma.dGx, &p->mma.dfx, &p->mma.dflags, &p->mma.dpx, &p->stream.dA, &p->stream.dtab,
                          &p->stream.dqx, &p->stream.dGx, &p->stream.dfx, &p->stream.dpx}) b->release();
    for (DevBuf &b : p->bp) b.release();
    p->dHsmall.release(); p->dHdense.release(); p->ddscr.release();
    p->repl.dHp.release(); p->repl.dtab.release(); p->repl.dcls.release(); p->repl.dX.release();
        for (auto &kv : p->flow_cfgs) kv.second.dsched.release();
        if (p->pinned_out) cudaFreeHost(p->pinned_out);
    }
    delete p;
}

extern "C" const char *modal_last_error(const modal_plan *p) { return p ? p->err.c_str() : g_create_error.c_str(); }

extern "C" modal_status modal_plan_query(const modal_plan *p, int what, void *dst, unsigned long long cap)
{
    if (!p || !dst) return MODAL_EINVAL;
    const modal_plan_desc &d = p->d;
    const int nq = d.n_q, cb = p->coeff_batch;
    auto put = [&](const void *src, size_t bytes) { if (bytes > cap) return MODAL_EINVAL; memcpy(dst, src, bytes); return MODAL_OK; };
    switch (what) {
        case MODAL_Q_MODE_M: return put(p->mq.m.data(), (size_t)nq * 4);
        case MODAL_Q_MODE_N: return put(p->mq.n.data(), (size_t)nq * 4);
        case MODAL_Q_PHI_M: return put(p->mphi.m.data(), p->mphi.m.size() * 4);
        case MODAL_Q_PHI_N: return put(p->mphi.n.data(), p->mphi.n.size() * 4);
        case MODAL_Q_LAMBDA: return put(p->mq.lambda.data(), (size_t)nq * 8);
        case MODAL_Q_OMEGA: return put(p->omega.data(), p->omega.size() * 8);
        case MODAL_Q_SIGMA: return put(p->sigma.data(), p->sigma.size() * 8);
        case MODAL_Q_NL_SCALE: return put(p->nl_scale.data(), p->nl_scale.size() * 8);
        case MODAL_Q_PICKUP: return put(p->pickup.data(), p->pickup.size() * 8);
        case MODAL_Q_ACTIVE: return put(p->active.data(), p->active.size() * 4);
        case MODAL_Q_COEFF_BATCH: return put(&cb, 4);
        case MODAL_Q_KERNEL_INFO: return put(p->kinfo, sizeof p->kinfo);
        case MODAL_Q_TILE_STATS: { const int ts[2] = {(int)p->tile_nz.size(), (int)p->nz_tiles}; return put(ts, sizeof ts); }
        case MODAL_Q_MMA_LAYOUT: {
            mh::MmaLayout L;
            int v[16] = {0};
            if (mma_host_layout(p, L)) {
                const int w[16] = {1, L.NKB, L.NGRP, L.NG, L.NC, L.S, L.RBT, L.RBQ, L.KC, L.KCL, L.G, L.rows_max,
                                   *std::min_element(L.kcnt.begin(), L.kcnt.end()), *std::max_element(L.kcnt.begin(), L.kcnt.end()),
                                   (int)(L.slab_bytes / 1024), *std::max_element(L.fcnt.begin(), L.fcnt.end())};
                memcpy(v, w, sizeof v);
            }
            return put(v, sizeof v);
        }
        case MODAL_Q_STREAM_LAYOUT: {
            mh::StreamLayout L;
            int v[16] = {0};
            if (stream_host_layout(p, 64, L)) {
                long long chunks = 0; for (const mh::StreamTile &t : L.tiles) chunks += t.nch;
                const int w[16] = {1, L.G, L.NKB, L.KC, (int)L.tiles.size(), L.tiles_max, *std::min_element(L.cta_ntiles.begin(), L.cta_ntiles.end()), L.bch_max,
                                   L.rows_max, *std::min_element(L.cta_rows.begin(), L.cta_rows.end()), L.nch_max, (int)chunks, (int)(L.a_bytes >> 20),
                                   *std::max_element(L.blk_nctas.begin(), L.blk_nctas.end()), 0, 0};
                memcpy(v, w, sizeof v);
            }
            return put(v, sizeof v);
        }
        case MODAL_Q_REPL_CHECK: {
            // host-side self check of the replicated-state kernel's layout on a grid of 132 CTAs (33 clusters of 4): rebuilds H^n[k][r]
            // from the packed blocks through the item descriptors (and their mirror images for the blocks stored once) and returns
            // {layout found, non-zero entries covered exactly once with the right value, non-zero entries of H, largest H of a CTA in KiB,
            //  most modes of a CTA, most rows of an item, packed floats in total, CTAs with a mode} as 8 doubles
            double out[8] = {0, 0, 0, 0, 0, 0, 0, 0};
            if (d.model == MODAL_VK && nq <= md::RP_THREADS) {
                const bool classes = d.geom == MODAL_RECT && p->opt.parity_order;
                auto cls_q = [&](int k_int) { const int k = p->perm[k_int]; return classes ? (p->mq.m[k] & 1) * 2 + (p->mq.n[k] & 1) : 0; };
                std::vector<int> class_start{0};
                for (int k = 1; k < nq; ++k) if (cls_q(k) != cls_q(k - 1)) class_start.push_back(k);
                class_start.push_back(nq);
                std::vector<double> Hi((size_t)d.n_phi * nq * nq);
                mh::unpack_flow_tiles(nq, d.n_phi, p->Hf, Hi.data());
                mh::ReplLayout L;
                if ((int)class_start.size() - 1 <= md::RP_MAXCLS && mh::repl_layout(nq, d.n_phi, 132, (size_t)212 * 256, class_start, Hi.data(), L)) {
                    out[0] = 1;
                    std::vector<unsigned char> seen(Hi.size(), 0);
                    double covered = 0, nonzero = 0, bad = 0;
                    for (double x : Hi) nonzero += x != 0.0;
                    int mm = 0;
                    for (int g = 0; g < L.G; ++g) {
                        const int *T = L.tab.data() + (size_t)g * mh::RP_CTA_STRIDE;
                        mm = std::max(mm, T[2]);
                        for (int t = 0; t < T[3]; ++t) {
                            const int *I = T + mh::RP_HDR + t * mh::RP_ITEM;
                            const int ld = I[1] & 0xffff, n = T[4 + (I[1] >> 16)];
                            for (int i = 0; i < I[3]; ++i)
                                for (int c = 0; c < 4; ++c) {
                                    const float v = L.Hp[L.cta_hoff[g] + I[0] + (size_t)i * ld + c];
                                    const int row = I[2] + i, col = I[4] + c;
                                    if (v == 0.f) continue;
                                    if (col >= nq) { bad += 1; continue; }
                                    for (int mirror = 0; mirror < (I[5] >= 0 ? 2 : 1); ++mirror) {
                                        const size_t e = ((size_t)n * nq + (mirror ? col : row)) * nq + (mirror ? row : col);
                                        if (seen[e] || (float)Hi[e] != v) bad += 1; else { seen[e] = 1; covered += 1; }
                                    }
                                }
                        }
                    }
                    out[1] = bad ? -bad : covered; out[2] = nonzero; out[3] = L.hfloats_max / 256.0; out[4] = mm; out[5] = L.rows_max;
                    out[6] = (double)L.Hp.size();
                    for (int g = 0; g < L.G; ++g) out[7] += L.cta_nmodes[g] > 0;
                }
            }
            return put(out, sizeof out);
        }
        case MODAL_Q_STREAM_CHECK: {
            // host-side self check of the H stream: rebuilds H^n[k][r] from the bf16 hi + lo chunks of every tile and returns
            // {non-zero entries covered, non-zero entries of H, max |hi + lo - H| / max |H|, rows owned in total} as 4 doubles
            mh::StreamLayout L;
            double out[4] = {0, 0, 0, 0};
            if (stream_host_layout(p, 64, L)) {
                std::vector<uint16_t> A;
                stream_host_A(p, L, A);
                std::vector<double> Hi((size_t)d.n_phi * nq * nq);
                mh::unpack_flow_tiles(nq, d.n_phi, p->Hf, Hi.data());
                double hmax = 0, emax = 0, covered = 0, nonzero = 0;
                for (double x : Hi) { hmax = std::max(hmax, std::fabs(x)); nonzero += x != 0.0; }
                std::vector<int> kop(L.KC * 16, -1);
                for (const mh::StreamBlock &b : L.blocks) for (int x = 0; x < b.nb; ++x) kop[b.koff + x] = b.k0 + x;
                for (const mh::StreamTile &t : L.tiles)
                    for (int u = 0; u < t.nch; ++u) {
                        const uint16_t *base = &A[(t.a_off + (size_t)u * 8192) / 2];
                        for (int kk = 0; kk < L.blocks[t.jb].nb; ++kk)
                            for (int e = 0; e < 16; ++e) {
                                const int r = kop[t.chunks[u] * 16 + e];
                                if (r < 0) continue;
                                const int o = mh::umma_chunk_off(kk, e) / 2;
                                const double v = (double)mh::bf16_to_float(base[o]) + (double)mh::bf16_to_float(base[2048 + o]);
                                const double h = Hi[((size_t)t.n * nq + L.blocks[t.jb].k0 + kk) * nq + r];
                                emax = std::max(emax, std::fabs(v - h));
                                covered += h != 0.0;
                            }
                    }
                double rows = 0; for (int x : L.cta_rows) rows += x;
                out[0] = covered; out[1] = nonzero; out[2] = hmax > 0 ? emax / hmax : 0; out[3] = rows;
            }
            return put(out, sizeof out);
        }
        case MODAL_Q_MMA_SLAB_CHECK: {
            // host-side self check of the operand packing: rebuilds H^n[k][r] from the bf16 hi + lo slabs of every CTA and
            // returns {entries covered, entries of H that are non-zero, max |hi + lo - H| / max |H|} as 3 doubles
            mh::MmaLayout L;
            double out[3] = {0, 0, 0};
            if (mma_host_layout(p, L)) {
                std::vector<uint16_t> slabs;
                mma_host_slabs(p, L, slabs);
                std::vector<double> Hi((size_t)d.n_phi * nq * nq);
                mh::unpack_flow_tiles(nq, d.n_phi, p->Hf, Hi.data());
                double hmax = 0, emax = 0, covered = 0, nonzero = 0;
                for (double x : Hi) { hmax = std::max(hmax, std::fabs(x)); nonzero += x != 0.0; }
                std::vector<int> kop(L.KP, -1);
                for (const mh::MmaBlock &b : L.blocks) for (int x = 0; x < b.nb; ++x) kop[b.koff + x] = b.k0 + x;
                for (int i = 0; i < L.NGRP; ++i)
                    for (int j = 0; j < L.NKB; ++j) {
                        const int c = i * L.NKB + j;
                        const uint16_t *base = &slabs[(size_t)c * L.slab_bytes / 2];
                        for (int x = 0; x < L.kcnt[c]; ++x)
                            for (int nl = 0; nl < L.NG; ++nl) {
                                const int n = L.nlist[(size_t)i * L.NG + nl];
                                if (n < 0) continue;
                                for (int kk = 0; kk < L.blocks[j].nb; ++kk)
                                    for (int e = 0; e < 16; ++e) {
                                        const int r = kop[L.klist[(size_t)c * L.KCL + x] * 16 + e];
                                        if (r < 0) continue;
                                        const size_t off = ((size_t)x * 2 * L.NC * 32 + mh::umma_chunk_off(nl * L.RBT + kk, e)) / 2;
                                        const double v = (double)mh::bf16_to_float(base[off]) + (double)mh::bf16_to_float(base[off + (size_t)L.NC * 16]);
                                        const double h = Hi[((size_t)n * nq + L.blocks[j].k0 + kk) * nq + r];
                                        emax = std::max(emax, std::fabs(v - h));
                                        covered += h != 0.0;
                                    }
                            }
                    }
                out[0] = covered; out[1] = nonzero; out[2] = hmax > 0 ? emax / hmax : 0.0;
            }
            return put(out, sizeof out);
        }
        case MODAL_Q_AIRY_ZETA4: return d.model == MODAL_VK ? put(p->zeta4.data(), p->zeta4.size() * 8) : MODAL_EINVAL;
        case MODAL_Q_H_FULL: {
            if (d.model != MODAL_VK) return MODAL_EINVAL;
            const size_t bytes = (size_t)d.n_phi * nq * nq * 8;
            if (bytes > cap) return MODAL_EINVAL;
            std::vector<double> Hi((size_t)d.n_phi * nq * nq);
            mh::unpack_flow_tiles(nq, d.n_phi, p->Hf, Hi.data());
            double *Hu = reinterpret_cast<double *>(dst);                      // internal -> user order
            for (int n = 0; n < d.n_phi; ++n)
                for (int a = 0; a < nq; ++a)
                    for (int b = 0; b < nq; ++b)
                        Hu[((size_t)n * nq + p->perm[a]) * nq + p->perm[b]] = Hi[((size_t)n * nq + a) * nq + b];
            return MODAL_OK;
        }
        default: return MODAL_EINVAL;
    }
}

extern "C" modal_status modal_derive_coeffs(const modal_plan *p, const modal_sample_geom *geom, double *omega,
                                            double *sigma, double *nl_scale, double *lambda, double *pickup)
{
    if (!p || !omega || !sigma) return MODAL_EINVAL;
    modal_sample_geom g = fill_geom(p, geom);
    derive_row(p, g, omega, sigma, nl_scale, lambda, pickup);
    return MODAL_OK;
}

extern "C" modal_status modal_project_bump(const modal_plan *p, double Lx, double Ly, double x0, double y0,
                                           double W, double A, double *q0)
{
    if (!p || !q0 || !(Lx > 0) || !(W > 0)) return MODAL_EINVAL;
    if (p->d.geom == MODAL_RECT) {
        if (!(Ly > 0)) return MODAL_EINVAL;
        mh::project_bump_rect(p->mq, Lx, Ly, x0, y0, W, A, q0);
    } else mh::project_bump_string(p->d.n_q, Lx, x0, W, A, q0);
    return MODAL_OK;
}

extern "C" modal_status modal_measure_peaks(int dev, modal_peaks *out)
{
    if (!out) return MODAL_EINVAL;
    memset(out, 0, sizeof *out);
#define PK(call) do { if ((call) != cudaSuccess) { cudaGetLastError(); rc = MODAL_ECUDA; goto done; } } while (0)
    modal_status rc = MODAL_OK;
    cudaDeviceProp prop{};
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    void *buf = nullptr, *small = nullptr;
    long long *cyc = nullptr;
    std::vector<long long> hc;
    float ms = 0;
    int sm = 0;
    const size_t big = (size_t)1 << 30;
    if (cudaSetDevice(dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) { cudaGetLastError(); return MODAL_ECUDA; }
    sm = prop.multiProcessorCount;
    PK(cudaEventCreate(&e0)); PK(cudaEventCreate(&e1));
    PK(cudaMalloc(&buf, big)); PK(cudaMalloc(&small, 1 << 16)); PK(cudaMalloc(&cyc, (size_t)sm * 8));
    PK(cudaMemset(buf, 1, big)); PK(cudaMemset(small, 0, 1 << 16));
    hc.resize(sm);
    {   // ---- FMA peaks: 8 CTAs of 256 threads per SM, 8 chains x 8 FMAs per iteration
        const int iters = 4096;
        auto run = [&](auto kern, auto x0, double &tf, double *clk) -> cudaError_t {
            kern<<<sm * 8, 256>>>(reinterpret_cast<decltype(x0) *>(small), 64, x0);                      // warm-up
            cudaEventRecord(e0); kern<<<sm * 8, 256>>>(reinterpret_cast<decltype(x0) *>(small), iters, x0); cudaEventRecord(e1);
            cudaError_t e = cudaEventSynchronize(e1);
            if (e != cudaSuccess) return e;
            cudaEventElapsedTime(&ms, e0, e1);
            const double fma = (double)sm * 8 * 256 * iters * 64.0;
            tf = 2.0 * fma / (ms * 1e-3) / 1e12;
            if (clk) *clk = fma / (ms * 1e-3) / ((double)sm * 128) / 1e6;                               // FP32: 128 FMA lanes per SM
            return cudaGetLastError();
        };
        PK(run(md::peak_fma_kernel<float>, 1.0f, out->fp32_tflops, &out->sm_clock_mhz));
        PK(run(md::peak_fma_kernel<double>, 1.0, out->fp64_tflops, nullptr));
    }
    {   // ---- read sweeps
        auto sweep = [&](size_t bytes, int passes, double &gbs) -> cudaError_t {
            md::peak_read_sweep_kernel<<<sm * 2, 512>>>(reinterpret_cast<const uint4 *>(buf), bytes / 16, 2, reinterpret_cast<unsigned *>(small));   // brings it into L2
            cudaEventRecord(e0);
            md::peak_read_sweep_kernel<<<sm * 2, 512>>>(reinterpret_cast<const uint4 *>(buf), bytes / 16, passes, reinterpret_cast<unsigned *>(small));
            cudaEventRecord(e1);
            cudaError_t e = cudaEventSynchronize(e1);
            if (e != cudaSuccess) return e;
            cudaEventElapsedTime(&ms, e0, e1);
            gbs = (double)bytes * passes / (ms * 1e-3) / 1e9;
            return cudaGetLastError();
        };
        PK(sweep((size_t)8 << 20, 400, out->l2_read_gbs_8mb));
        PK(sweep((size_t)64 << 20, 50, out->l2_read_gbs_64mb));
        PK(sweep(big, 4, out->hbm_read_gbs));
    }
    {   // ---- shared memory
        const int iters = 4096;
        PK(cudaFuncSetAttribute(md::peak_smem_read_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536));
        md::peak_smem_read_kernel<<<sm, 512, 65536>>>(64, cyc, reinterpret_cast<unsigned *>(small));
        cudaEventRecord(e0); md::peak_smem_read_kernel<<<sm, 512, 65536>>>(iters, cyc, reinterpret_cast<unsigned *>(small)); cudaEventRecord(e1);
        PK(cudaEventSynchronize(e1));
        cudaEventElapsedTime(&ms, e0, e1);
        PK(cudaMemcpy(hc.data(), cyc, (size_t)sm * 8, cudaMemcpyDeviceToHost));
        double c = 0; for (int i = 0; i < sm; ++i) c += (double)hc[i];
        out->smem_bytes_per_clk_sm = 65536.0 * iters / (c / sm);
        out->smem_read_gbs = 65536.0 * iters * sm / (ms * 1e-3) / 1e9;
    }
    {   // ---- TMEM
        const int iters = 256;
        md::peak_tmem_read_kernel<<<sm, 128>>>(8, cyc, reinterpret_cast<unsigned *>(small));
        md::peak_tmem_read_kernel<<<sm, 128>>>(iters, cyc, reinterpret_cast<unsigned *>(small));
        PK(cudaDeviceSynchronize());
        PK(cudaMemcpy(hc.data(), cyc, (size_t)sm * 8, cudaMemcpyDeviceToHost));
        double c = 0; for (int i = 0; i < sm; ++i) c += (double)hc[i];
        out->tmem_read_bytes_per_clk_sm = 128.0 * 512 * 4 * iters / (c / sm);
    }
    {   // ---- exchange hops (one-way = half a round trip)
        const int rounds = 2000;
        double *dst[4] = {&out->hop_cycles_idle, &out->hop_cycles_loaded, &out->relacq_hop_cycles_idle, &out->relacq_hop_cycles_loaded};
        for (int v = 0; v < 4; ++v) {
            const int mode = v >> 1, load = v & 1;
            PK(cudaMemset(small, 0, 1 << 16));
            char *sb = reinterpret_cast<char *>(small);
            md::peak_hop_kernel<<<sm, 512>>>(reinterpret_cast<unsigned long long *>(sb), reinterpret_cast<unsigned *>(sb + 4096), rounds, mode, load,
                                             reinterpret_cast<const uint4 *>(buf), ((size_t)32 << 20) / 16, reinterpret_cast<volatile int *>(sb + 8192),
                                             cyc, reinterpret_cast<unsigned *>(sb + 8256));
            PK(cudaDeviceSynchronize());
            PK(cudaMemcpy(hc.data(), cyc, 8, cudaMemcpyDeviceToHost));
            *dst[v] = hc[0] > 0 ? (double)hc[0] / rounds / 2.0 : -1.0;
        }
    }
done:
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (buf) cudaFree(buf);
    if (small) cudaFree(small);
    if (cyc) cudaFree(cyc);
#undef PK
    return rc;
}
