// planner.cpp -- S1 of the hot path: the host-side tile scheduler (successor of the paper's
// hclMatrixPartitioner).  Pure host arithmetic; needs no GPU.
//
// The paper's rule (one B slice, two A slices and two C blocks fit the device; equal slices; :289,
// example :301) is kept as hclMatrixPartitioner().  hclooc_plan() generalises it:
//   * ragged edge slices (ceil division) instead of equal slices only,
//   * n_sets >= 2 (A slice, C block) buffer pairs so several small steps can be in flight,
//   * an optional second B slice buffer so the next B slice is prefetched in chunks under compute
//     (the paper reloads B un-overlapped at i == h-1, :236-242),
//   * an optional split of K into panels when even the thinnest B slice does not fit,
// and picks among the feasible candidates with a small cost model:
//     T = max(link path, compute path) + tail,   link = host<->device bytes at measured bandwidth,
//     compute = 2MNK at the measured DMMA rate, de-rated by tile padding and SM fill.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include "internal.h"

namespace hclooc {

namespace {
double env_or(const char* name, double dflt) {
    const char* s = std::getenv(name);
    if (!s || !*s) return dflt;
    char* end = nullptr;
    double v = std::strtod(s, &end);
    return (end && end != s && v > 0) ? v : dflt;
}
int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }
int64_t round_up(int64_t a, int64_t b) { return ceil_div(a, b) * b; }
constexpr int64_t TILE = 128;          // CTA tile edge of the S5 kernel
constexpr int64_t LD_ALIGN = 16;       // device leading dimensions are multiples of 16 doubles (128 B)
constexpr uint64_t BUF_ALIGN = 1024;   // every device buffer starts on a 1 KiB boundary
constexpr int NUM_SMS = 148;
constexpr double OVERLAP_PENALTY = 0.02;   // measured: with the link 70 % busy under a compute-bound plan nothing is lost (config 3, w = 10)
constexpr double STREAMK_MIN_TILES = 32;
}  // namespace

namespace {
MachineModel& model_storage() {
    static MachineModel mm = {
        env_or("HCLOOC_FP64_TFLOPS", 37.17) * 1e12,   // DMMA loop, 148 SMs, sustained (profiles/r01_box_probe.md)
        env_or("HCLOOC_H2D_GBPS", 55.5) * 1e9,        // link rates of the first box probed; hclooc_calibrate_link() replaces them with
        env_or("HCLOOC_D2H_GBPS", 51.5) * 1e9,        // what THIS box measures (the boxes of the pool differ: 51.5-57 D2H, 88-100 duplex)
        env_or("HCLOOC_DUPLEX_GBPS", 88.0) * 1e9,
        env_or("HCLOOC_COPY_LATENCY_US", 8.0) * 1e-6, // per copy inside the pipeline (event waits between copies); 4-5 us back to back
        env_or("HCLOOC_LAUNCH_LATENCY_US", 5.0) * 1e-6,
    };
    return mm;
}
}  // namespace

const MachineModel& machine_model() { return model_storage(); }

// measured link rates replace the defaults (not a rate the environment pins)
void set_machine_link(double h2d_Bps, double d2h_Bps, double duplex_Bps) {
    MachineModel& mm = model_storage();
    if (!std::getenv("HCLOOC_H2D_GBPS") && h2d_Bps > 1e9) mm.h2d_Bps = h2d_Bps;
    if (!std::getenv("HCLOOC_D2H_GBPS") && d2h_Bps > 1e9) mm.d2h_Bps = d2h_Bps;
    if (!std::getenv("HCLOOC_DUPLEX_GBPS") && duplex_Bps > 1e9) mm.duplex_Bps = duplex_Bps;
}

int g_direct_max_cluster = 16;      // what direct_max_cluster() found on the device (set by the executor); 16 on a B200
void set_planner_max_cluster(int n) { g_direct_max_cluster = n >= 16 ? 16 : 8; }

namespace {

struct Cand {
    int64_t mb, nb, kb, h, w, kpanels;
    int n_sets, n_abuf, n_bbuf, ksplit, n_scratch;
    bool ta;              // A is stored K x M: its slices are uploaded as kb rows of mb doubles (narrow rows when mb is small)
    bool c_dev;           // C lives in device memory: its block copies are device-to-device, not host-link traffic
    bool c_in_host;       // ... except the uploads of K panel 0, which read the initial C from a HOST matrix (operands_on_device = 5)
    int64_t lda_dev, ldb_dev, ldc_dev;
    uint64_t a_bytes, b_bytes, c_bytes, ws_bytes;
    uint64_t bytes_h2d, bytes_d2h, n_h2d, n_d2h;
    double t_flop, t_link, t_model;
};

// Budget share kept free for the two stream-K scratch buffers (only when that is at most 5 % of the budget).
uint64_t streamk_reserve(uint64_t budget) {
    const uint64_t need = 2 * (uint64_t)streamk_scratch_bytes();
    return need * 20 <= budget ? need : 0;
}

// Exact host<->device traffic of the schedule the executor builds from this candidate (executor.cu
// build_schedule): columns of blocks in order, rows in serpentine order, A slices in an LRU cache of
// n_abuf buffers -- so at every column switch inside a K panel the min(n_abuf, h) slices at the turning
// end are reused, not uploaded again.
void fill_traffic(Cand& c, int64_t M, int64_t N, int64_t K, bool beta_nz, bool scale_only) {
    const uint64_t MN = (uint64_t)M * (uint64_t)N;
    const uint64_t steps = (uint64_t)c.h * c.w * c.kpanels;
    uint64_t el_h2d = 0, n_h2d = 0;
    if (!scale_only) {
        const int64_t reuse = std::min<int64_t>(c.n_abuf, c.h);                 // slices reused per column switch
        const int64_t rows_top = std::min<int64_t>(M, reuse * c.mb);            // rows of the first `reuse` slices
        const int64_t rows_bottom = M - (c.h - reuse) * c.mb;                   // rows of the last `reuse` slices
        // per K panel p (depth kk_p): column 0 uploads every slice, column j >= 1 (slab sl = p*w + j) keeps the slices at
        // the end where column sl-1 stopped: the bottom when sl-1 is even (it ran downwards), the top otherwise.
        // Closed form over the panels: all but the last are kb deep.
        const int64_t kk_last = K - (c.kpanels - 1) * c.kb;
        auto panel_cols = [&](int64_t p, int64_t* n_top, int64_t* n_bottom) {   // columns j = 1..w-1 of panel p by turning end
            const int64_t first = p * c.w + 1, last = p * c.w + c.w - 1;            // slabs sl; parity of sl-1 decides
            if (last < first) { *n_top = *n_bottom = 0; return; }
            const int64_t n = last - first + 1;
            const int64_t n_odd_prev = ((first - 1) & 1) ? (n + 1) / 2 : n / 2;    // sl-1 odd -> kept = rows_top
            *n_top = n_odd_prev; *n_bottom = n - n_odd_prev;
        };
        for (int pass = 0; pass < 2; ++pass) {
            // pass 0: the kpanels-1 full panels (their column parities alternate with p*w, so count panel by panel only
            // when w is odd; for even w every panel looks the same), pass 1: the last panel
            if (pass == 0) {
                const int64_t full = c.kpanels - 1;
                if (full <= 0) continue;
                int64_t nt = 0, nbm = 0;
                if (c.w % 2 == 0) { panel_cols(0, &nt, &nbm); nt *= full; nbm *= full; }
                else {
                    int64_t t0, b0, t1, b1;
                    panel_cols(0, &t0, &b0); panel_cols(1, &t1, &b1);
                    const int64_t even_p = (full + 1) / 2, odd_p = full / 2;
                    nt = t0 * even_p + t1 * odd_p; nbm = b0 * even_p + b1 * odd_p;
                }
                el_h2d += (uint64_t)full * (uint64_t)M * c.kb + (uint64_t)(nt * (M - rows_top) + nbm * (M - rows_bottom)) * c.kb;
                n_h2d += (uint64_t)full * c.h + (uint64_t)(nt + nbm) * (c.h - reuse);
            } else {
                int64_t nt, nbm;
                panel_cols(c.kpanels - 1, &nt, &nbm);
                el_h2d += (uint64_t)M * kk_last + (uint64_t)(nt * (M - rows_top) + nbm * (M - rows_bottom)) * kk_last;
                n_h2d += (uint64_t)c.h + (uint64_t)(nt + nbm) * (c.h - reuse);
            }
        }
        el_h2d += (uint64_t)K * (uint64_t)N;                                    // every B slice once
        const uint64_t slabs = (uint64_t)c.w * c.kpanels;
        if (c.n_bbuf == 1) n_h2d += slabs;
        else {
            n_h2d += 1;                                                         // first slice in one piece
            // prefetched slices sl = 1 .. slabs-1: those of the last panel are kk_last deep, the others kb
            int64_t i0, nch_full, nch_last;
            prefetch_layout(c.h, c.kb, c.n_sets, &i0, &nch_full);
            prefetch_layout(c.h, kk_last, c.n_sets, &i0, &nch_last);
            const uint64_t in_last = (c.kpanels > 1) ? (uint64_t)c.w : (uint64_t)c.w - 1;   // slabs >= 1 inside the last panel
            n_h2d += in_last * (uint64_t)nch_last + (slabs - 1 - in_last) * (uint64_t)nch_full;
        }
    }
    const uint64_t MNlink = c.c_dev ? 0 : MN;                                   // copies are still enqueued, bytes are not link bytes
    if (beta_nz) { el_h2d += c.c_in_host ? MN : MNlink; n_h2d += (uint64_t)c.h * c.w; }
    if (c.kpanels > 1) { el_h2d += (uint64_t)(c.kpanels - 1) * MNlink; n_h2d += (uint64_t)(c.kpanels - 1) * c.h * c.w; }
    c.bytes_h2d = 8 * el_h2d;
    c.n_h2d = n_h2d;
    c.bytes_d2h = 8 * (uint64_t)c.kpanels * MNlink;
    c.n_d2h = steps;
}

void cost(Cand& c, int64_t M, int64_t N, int64_t K, bool beta_nz, bool scale_only, const MachineModel& mm, uint64_t budget) {
    fill_traffic(c, M, N, K, beta_nz, scale_only);
    const double steps = (double)c.h * c.w * c.kpanels;
    const double flops = scale_only ? 0.0 : 2.0 * (double)M * (double)N * (double)K;
    // tile padding and SM fill
    const double tiles_step = (double)ceil_div(c.mb, TILE) * (double)ceil_div(c.nb, TILE);
    // exact share of useful work in the 128 x 128 tiles the kernel launches (ragged last slices included)
    const int64_t m_last = M - (c.h - 1) * c.mb, n_last = N - (c.w - 1) * c.nb;
    const double tile_rows = (double)((c.h - 1) * ceil_div(c.mb, TILE) + ceil_div(m_last, TILE));
    const double tile_cols = (double)((c.w - 1) * ceil_div(c.nb, TILE) + ceil_div(n_last, TILE));
    const double pad_eff = ((double)M * (double)N) / (tile_rows * tile_cols * (double)(TILE * TILE));
    // too few tiles in flight to fill the SMs: a cluster of 2 or 4 CTAs shares each tile's K range.  When the
    // link is the bound the kernels of successive steps hardly overlap, so one step's tiles are all there is.
    static const int force_ks = (int)env_or("HCLOOC_FORCE_KSPLIT", 0);
    c.t_flop = flops / mm.fp64_flops;
    const double t_in = c.bytes_h2d / mm.h2d_Bps + c.n_h2d * mm.copy_latency_s;
    const double t_out = c.bytes_d2h / mm.d2h_Bps + c.n_d2h * mm.copy_latency_s;
    double t_in_rows = 0.0;
    const double a_row_factor = (c.ta && !scale_only && c.mb * 8 < 2048) ? 1.0 + 0.45 * (2048.0 / (double)(c.mb * 8) - 1.0) : 1.0;
    if (c.ta && !scale_only && c.mb * 8 < 2048) {
        // 2-D copies run at full rate only from ~2 KiB per row up, and the slices of a transposed A have rows of mb
        // doubles.  Measured on config 2 with A^T: 1 KiB rows (mb = 128) move at ~35 GB/s inside the pipeline, 2 KiB rows
        // within 1.3 % of the untransposed call; alone, 128-byte rows reach 8.3 GB/s (profiles/r01_box_probe.md).
        const double a_bytes_all = (double)c.bytes_h2d - 8.0 * (double)K * (double)N - ((beta_nz || c.kpanels > 1) && !c.c_dev ? 8.0 * (double)M * (double)N * (beta_nz ? c.kpanels : c.kpanels - 1) : 0.0) -
                                   (beta_nz && c.c_dev && c.c_in_host ? 8.0 * (double)M * (double)N : 0.0);
        t_in_rows = std::max(0.0, a_bytes_all) / mm.h2d_Bps * 0.45 * (2048.0 / (double)(c.mb * 8) - 1.0);
    }
    c.t_link = std::max(std::max(t_in + t_in_rows, t_out), (double)(c.bytes_h2d + c.bytes_d2h) / mm.duplex_Bps + t_in_rows);
    const bool link_bound = c.t_link > c.t_flop / std::max(1e-3, pad_eff);
    const double steps_in_flight = link_bound ? 1.0 : (double)std::max(1, c.n_sets - 2);
    c.ksplit = scale_only ? 1 : (force_ks ? force_ks : dgemm_auto_ksplit((int64_t)(steps_in_flight * tiles_step), c.kb));
    // Optional (HCLOOC_STREAMK_STEPS=1): compute-bound plans run every step as ONE persistent stream-K launch on
    // all SMs, two compute streams alternating; costs two scratch buffers inside the budget and ~10 us per step.
    // Measured on config 4: 0.969 of the FP64 peak against 0.976 for well-shaped steps whose one-CTA-per-tile
    // kernels overlap on several streams, so it is not the default.
    static const bool streamk_steps = std::getenv("HCLOOC_STREAMK_STEPS") != nullptr;   // off by default: measured 0.7 % behind
    const bool want_streamk = streamk_steps && !scale_only && !link_bound && !force_ks && tiles_step >= STREAMK_MIN_TILES &&
                              c.kb >= 256 && streamk_reserve(budget) > 0 && c.ws_bytes + streamk_reserve(budget) <= budget;
    c.n_scratch = want_streamk ? 2 : 0;
    if (want_streamk) c.ksplit = -1;
    const double in_flight = want_streamk ? (double)NUM_SMS : std::max(1, c.n_sets - 2) * tiles_step * c.ksplit;
    double fill = std::min(1.0, in_flight / NUM_SMS);
    if (!want_streamk && tiles_step >= NUM_SMS) fill = std::min(fill, 0.98);
    if (!want_streamk && fill >= 1.0 && tiles_step < NUM_SMS) fill = 0.975;     // measured: kernels of several steps interleave imperfectly
    if (!want_streamk && c.n_sets < 4) fill *= (c.n_sets == 2 ? 0.96 : 0.985);  // too few C blocks in flight to fill the wave tails
    const double t_compute = c.t_flop / std::max(1e-3, pad_eff * fill) + steps * (want_streamk ? 10e-6 : 1e-6);
    const bool cload = beta_nz || c.kpanels > 1;
    const double t_pro = ((double)c.b_bytes + (double)c.a_bytes + (cload ? (double)c.c_bytes : 0.0)) / mm.h2d_Bps + 3 * mm.copy_latency_s;
    // one step's kernel running alone: what the link waits for when a column drains, and the tail of the call
    const double sms_step = c.ksplit < 0 ? (double)NUM_SMS : std::min<double>(NUM_SMS, tiles_step * c.ksplit);
    const double t_kernel = (flops / std::max(1.0, steps)) / (mm.fp64_flops * sms_step / NUM_SMS) + mm.launch_latency_s;
    // Column by column: the first column of a K panel uploads every A slice, the later ones only what the cache
    // lost, so the link demand is front-loaded -- a plan with many thin columns is link-bound in its first column
    // even when the whole call is compute-bound (measured: config 4 with 47 columns lost 2 % there).
    const double n_cols = (double)c.w * c.kpanels;
    const double comp_col = t_compute / n_cols;
    const double a_first = scale_only ? 0.0 : 8.0 * (double)M * (double)c.kb;
    const double mn_link = c.c_dev ? 0.0 : 8.0 * (double)M * (double)N;
    const double mn_up0 = (c.c_dev && c.c_in_host) ? 8.0 * (double)M * (double)N : mn_link;      // C uploads of K panel 0
    const double a_all = (double)c.bytes_h2d - 8.0 * (double)K * (double)N - (beta_nz ? mn_up0 : 0.0) -
                         (c.kpanels > 1 ? (double)(c.kpanels - 1) * mn_link : 0.0);
    const double a_later = n_cols > c.kpanels ? std::max(0.0, a_all - a_first * c.kpanels) / (n_cols - c.kpanels) : 0.0;
    const double c_col = c.c_dev ? 0.0 : 8.0 * (double)M * (double)c.nb;
    const double c_col_up = (c.c_dev && c.c_in_host && c.kpanels == 1) ? 8.0 * (double)M * (double)c.nb : c_col;
    auto link_col = [&](double a_bytes) {
        const double up = a_bytes * a_row_factor + (scale_only ? 0.0 : (double)c.b_bytes) + (cload ? c_col_up : 0.0);
        const double lat = (double)c.h * 2.0 * mm.copy_latency_s;
        return std::max(std::max(up / mm.h2d_Bps, c_col / mm.d2h_Bps), (up + c_col) / mm.duplex_Bps) + lat;
    };
    double stall_comp = 0.0, stall_link = 0.0;      // per column switch, with a single B buffer
    if (c.n_bbuf == 1) {
        stall_comp = (double)c.b_bytes / mm.h2d_Bps;                  // compute idles while the next B slice loads
        // the link idles (a) while the last kernels of a column drain before S(b_j) may overwrite the buffer,
        // less the uploads issued ahead of the reload, and (b) after the reload once every C buffer is held by
        // a step whose kernel has only just started
        const double t_up = ((double)c.bytes_h2d - 8.0 * (double)K * (double)N) / std::max(1.0, steps) / mm.h2d_Bps + mm.copy_latency_s;
        const double c_rate_up = (c.c_dev && !c.c_in_host) ? 1.0e12 : mm.h2d_Bps, c_rate_down = c.c_dev ? 1.0e12 : mm.d2h_Bps;
        const double t_cup = cload ? (double)c.c_bytes / c_rate_up + mm.copy_latency_s : t_up;
        const double pre = (double)early_uploads(c.h, c.n_sets, c.n_abuf);
        const double drain = std::max(0.0, t_kernel - pre * t_cup);
        const double refill = std::max(0.0, t_kernel + (double)c.c_bytes / c_rate_down - std::max(0.0, c.n_sets - pre - 1.0) * t_up);
        stall_link = drain + refill;
    }
    const double l_first = link_col(a_first), l_later = link_col(a_later);
    const double body = c.kpanels * std::max(comp_col + stall_comp, l_first + stall_link) +
                        (n_cols - c.kpanels) * std::max(comp_col + stall_comp, l_later + stall_link);
    const double comp_path = t_pro + t_compute, link_path = c.t_link;
    const double t_tail = t_kernel + (double)c.c_bytes / mm.d2h_Bps + mm.copy_latency_s;
    // imperfect overlap: the shorter path still costs a fraction of its length (bursty uploads, shared
    // DMA/HBM resources), which also keeps plans away from the edge where link time ~ compute time
    c.t_model = t_pro + body + OVERLAP_PENALTY * std::min(comp_path, link_path) + t_tail + mm.launch_latency_s;
    // between near-equal plans take the one whose slices are whole tiles: padded tiles burn FP64 issue slots and
    // power for nothing even when the link hides their time
    c.t_model *= 1.0 + 0.3 * (1.0 - (double)N / (tile_cols * (double)TILE));     // column padding only: rows pad with mb < 128 by design
}

}  // namespace
}  // namespace hclooc

using namespace hclooc;

extern "C" int hclooc_plan(int64_t M, int64_t N, int64_t K, int beta_nonzero, int alpha_zero,
                           size_t device_budget_bytes, hclooc_plan_t* out) {
    return hclooc_plan_ex(M, N, K, beta_nonzero, alpha_zero, device_budget_bytes, 0, out);
}

extern "C" int hclooc_plan_ex(int64_t M, int64_t N, int64_t K, int beta_nonzero, int alpha_zero,
                              size_t device_budget_bytes, int operands_on_device, hclooc_plan_t* out) {
    return plan_impl(M, N, K, beta_nonzero, alpha_zero, device_budget_bytes, operands_on_device, 0, 0, out);
}

// transa / transb (hclooc_dgemm_t): the device slices keep the layout the operand is stored in -- an A slice is kb x mb
// (leading dimension lda_dev >= mb), a B slice nb x kb (ldb_dev >= kb) -- which only changes the buffer sizes here.
int hclooc::plan_impl(int64_t M, int64_t N, int64_t K, int beta_nonzero, int alpha_zero, size_t device_budget_bytes,
                      int operands_on_device, int transa, int transb, hclooc_plan_t* out) {
    const MachineModel& mm = machine_model();
    const bool c_dev = operands_on_device == 2 || operands_on_device == 5, c_in_host = operands_on_device == 5;
    const bool direct_ok = operands_on_device == 3 || operands_on_device == 4, direct_forced = operands_on_device == 4;
    if (operands_on_device >= 2) operands_on_device = 0;
    if (M < 0) return -1;
    if (N < 0) return -2;
    if (K < 0) return -3;
    if (!out) return operands_on_device ? -8 : -7;
    std::memset(out, 0, sizeof(*out));
    out->M = M; out->N = N; out->K = K;
    out->beta_nonzero = beta_nonzero ? 1 : 0;
    const bool scale_only = (alpha_zero != 0) || (K == 0);
    out->scale_only = scale_only ? 1 : 0;
    if (scale_only) transa = transb = 0;
    out->trans = (transa ? 1 : 0) | (transb ? 2 : 0);
    if (M == 0 || N == 0) return HCLOOC_OK;                       // nothing to do: zero steps
    if (operands_on_device) {
        // the in-core case (the switch to out-of-core happens only when the matrices do not
        // fit): nothing to stage, one DGEMM over the caller's matrices, no workspace
        out->mb = M; out->nb = N; out->kb = scale_only ? 0 : K;
        out->h = out->w = out->kpanels = out->n_steps = 1;
        out->ksplit = scale_only ? 1 : dgemm_auto_ksplit(dgemm_tile_count(M, N), K);
        out->flops = scale_only ? 0.0 : 2.0 * (double)M * (double)N * (double)K;
        out->t_flop_s = out->flops / mm.fp64_flops;
        out->t_model_s = out->t_flop_s + mm.launch_latency_s;
        return HCLOOC_OK;
    }
    const bool beta_nz = beta_nonzero != 0;
    const int64_t Keff = scale_only ? 0 : K;
    const uint64_t S = (uint64_t)device_budget_bytes;

    // experiment knobs (not part of the ABI): force parts of the plan
    const int64_t force_nb = (int64_t)env_or("HCLOOC_FORCE_NB", 0), force_mb = (int64_t)env_or("HCLOOC_FORCE_MB", 0);
    const int force_sets = (int)env_or("HCLOOC_FORCE_SETS", 0), force_bbuf = (int)env_or("HCLOOC_FORCE_BBUF", 0);
    const int64_t force_abuf = (int64_t)env_or("HCLOOC_FORCE_ABUF", 0);
    bool found = false;
    Cand best{};
    static const int set_choices[] = {2, 3, 4, 5, 6, 7, 8, 10, 12};
    for (int64_t kpanels = 1; kpanels <= std::max<int64_t>(1, ceil_div(Keff, 16)) && !found; kpanels *= 2) {
        const int64_t kb = scale_only ? 0 : std::min(Keff, round_up(ceil_div(Keff, kpanels), 16));
        const int64_t kp = scale_only ? 1 : ceil_div(Keff, kb);
        int64_t last_nb = -1;
        const int64_t wmax = ceil_div(N, 16);
        for (int64_t wi = 2; wi <= 2 * wmax + 1; wi = (wi < 128 ? wi + 1 : wi + wi / 8)) {
            // two slice widths per w: the thinnest multiple of 16 and the thinnest multiple of the tile edge
            const int64_t w = wi / 2;
            const int64_t nb = std::min(N, round_up(ceil_div(N, w), (wi & 1) ? TILE : 16));
            if (nb == last_nb) continue;
            last_nb = nb;
            if (force_nb && nb != std::min(N, round_up(force_nb, 16))) continue;
            const int64_t weff = ceil_div(N, nb);
            const int64_t lda_dev = round_up(std::max<int64_t>(kb, 1), LD_ALIGN);      // A as stored M x K; A^T: set per candidate
            const int64_t ldc_dev = round_up(nb, LD_ALIGN);
            const int64_t ldb_dev = transb ? round_up(std::max<int64_t>(kb, 1), LD_ALIGN) : ldc_dev;
            const uint64_t b_bytes = scale_only ? 0 : round_up((uint64_t)(transb ? nb : kb) * ldb_dev * 8, BUF_ALIGN);
            for (int n_bbuf = 1; n_bbuf <= (scale_only || weff * kp == 1 ? 1 : 2); ++n_bbuf) {
                if ((uint64_t)n_bbuf * b_bytes >= S) continue;
                if (force_bbuf && n_bbuf != force_bbuf && !(scale_only || weff * kp == 1)) continue;
                const uint64_t rem = S - (uint64_t)n_bbuf * b_bytes;
                const uint64_t per_row = 8 * (uint64_t)((scale_only ? 0 : lda_dev) + ldc_dev);
                for (int n_sets : set_choices) {
                    if (force_sets && n_sets != force_sets) continue;
                    const uint64_t overhead = (uint64_t)n_sets * 2 * BUF_ALIGN;
                    if (rem <= overhead) continue;
                    const int64_t rows_max = (int64_t)((rem - overhead) / per_row / n_sets);
                    if (rows_max < 1) continue;
                    // row-count candidates: as many as fit, or a few standard sizes below that
                    int64_t tried[6];
                    int nt = 0;
                    int64_t top = std::min(M, rows_max);
                    if (top >= TILE) top = top / TILE * TILE; else if (top >= 16 && transa) top = top / 16 * 16; else if (top >= 8) top = top / 8 * 8;
                    tried[nt++] = top;
                    for (int64_t cand_mb : {(int64_t)1024, (int64_t)512, (int64_t)256, (int64_t)128})
                        if (cand_mb < top) tried[nt++] = cand_mb;
                    if (force_mb) { nt = 0; if (force_mb <= std::min(M, rows_max)) tried[nt++] = force_mb; }
                    // a call that fills a resident panel of a look-ahead routine (C read from the host, stored on the device:
                    // hclooc_dpotrf, hclooc_dtrsm[_side]) shares the SMs with that routine's device phase on other streams; the model
                    // sees a link-bound call and would cut it into 128-row steps of split-K clusters.  Measured (32768^2, 4 GiB): blocks
                    // of 1024 rows make the Cholesky (tall panels: M = 4096..28672) 4.7 % and the right-side DTRSM (M = 32768) 2 % faster;
                    // the left-side DTRSM fills block ROWS (M = NB = 4096, N wide), where 1024-row blocks leave 4 steps per column and
                    // cost 4 %: the floor is a sixteenth of M, at most 1024.
                    const int64_t mb_floor = (c_in_host && !force_mb) ? std::min<int64_t>(top, std::min<int64_t>(1024, std::max<int64_t>(128, M / 16 / 128 * 128))) : 0;
                    for (int q = 0; q < nt; ++q) {
                        if (tried[q] < mb_floor) continue;
                        Cand c{};
                        c.c_dev = c_dev;
                        c.c_in_host = c_in_host;
                        c.ta = transa != 0;
                        c.mb = tried[q]; c.nb = nb; c.kb = kb; c.kpanels = kp;
                        c.h = ceil_div(M, c.mb); c.w = weff;
                        c.n_sets = (int)std::min<int64_t>(n_sets, std::max<int64_t>(2, c.h * c.w * kp));
                        c.n_bbuf = n_bbuf;
                        c.lda_dev = scale_only ? 0 : (transa ? round_up(c.mb, LD_ALIGN) : lda_dev);
                        c.ldb_dev = scale_only ? 0 : ldb_dev; c.ldc_dev = ldc_dev;
                        c.a_bytes = scale_only ? 0 : round_up((uint64_t)(transa ? kb * c.lda_dev : c.mb * lda_dev) * 8, BUF_ALIGN);
                        c.b_bytes = b_bytes;
                        c.c_bytes = round_up((uint64_t)c.mb * ldc_dev * 8, BUF_ALIGN);
                        c.n_abuf = scale_only ? 0 : c.n_sets;
                        c.ws_bytes = (uint64_t)n_bbuf * b_bytes + (uint64_t)c.n_sets * (c.a_bytes + c.c_bytes);
                        if (c.ws_bytes > S) continue;
                        if (!scale_only && c.w > 1 && c.a_bytes > 0) {
                            // spare budget holds more A slices: more reuse at every column switch
                            const uint64_t room = S - c.ws_bytes > streamk_reserve(S) ? S - c.ws_bytes - streamk_reserve(S) : 0;
                            const int64_t extra = std::min<int64_t>((int64_t)(room / c.a_bytes), std::max<int64_t>(0, c.h - c.n_abuf));
                            const int64_t capped = std::min<int64_t>(extra, force_abuf ? std::max<int64_t>(0, force_abuf - c.n_abuf) : 256 - c.n_abuf);
                            if (capped > 0) { c.n_abuf += (int)capped; c.ws_bytes += (uint64_t)capped * c.a_bytes; }
                        }
                        cost(c, M, N, Keff, beta_nz, scale_only, mm, S);
                        c.ws_bytes += (uint64_t)c.n_scratch * streamk_scratch_bytes();
                        const double steps = (double)c.h * c.w * c.kpanels, bsteps = (double)best.h * best.w * best.kpanels;
                        if (!found || c.t_model < best.t_model * (1 - 1e-9) ||
                            (c.t_model <= best.t_model * (1 + 1e-9) && steps < bsteps)) {
                            best = c;
                            found = true;
                        }
                    }
                }
            }
        }
    }
    // ---- DIRECT mode: no staging, one launch whose tiles read A and B from host memory through TMA and update C in
    // place over the link.  Measured (profiles/r01_direct_mode.md): SM-initiated reads of pinned host memory run at
    // ~50 GB/s with no reuse between tiles in L2, so the time is the sum of every tile's own reads over that rate
    // plus ~30 us fixed -- better than a staged plan only where that one is bound by per-copy latency.
    if (direct_ok && M <= 0x7fffffffLL && N <= 0x7fffffffLL && K <= 0x7fffffffLL) {
        const double tm = (double)ceil_div(M, TILE), tn = (double)ceil_div(N, TILE);
        // the tiles of a cluster share their loads by TMA multicast (dgemm_direct_sm100.cu): A crosses the link once per
        // cluster column, B once per cluster row; transposed operands use the plain tile kernel (no sharing)
        int cm = 1, cn = 1;
        if (!transa && !transb && !scale_only) direct_cluster_shape(M, N, g_direct_max_cluster, &cm, &cn);
        out->direct_cm = cm; out->direct_cn = cn;
        const double rd = 8.0 * ((scale_only ? 0.0 : std::ceil(tn / cn) * (double)M * (double)Keff + std::ceil(tm / cm) * (double)Keff * (double)N) +
                                 (beta_nz ? (double)M * (double)N : 0.0));
        const double wr = 8.0 * (double)M * (double)N;
        // measured: 46-50 GB/s when every tile loads for itself; through multicasting clusters (their CTAs advance in
        // lockstep, a stage at a time) 24-36 GB/s with one cluster in flight, 35 with four, 44 with 64
        const double n_clusters = std::ceil(tm / cm) * std::ceil(tn / cn);
        const double direct_Bps = env_or("HCLOOC_DIRECT_GBPS", cm * cn > 1 ? std::min(45.0, 30.0 + 3.5 * std::sqrt(n_clusters)) : 50.0) * 1e9;
        const double t_link = std::max(std::max(rd / direct_Bps, wr / mm.d2h_Bps), (rd + wr) / mm.duplex_Bps);
        const double t_flop = (scale_only ? 0.0 : 2.0 * (double)M * (double)N * (double)Keff) / mm.fp64_flops;
        const double waves = std::ceil(tm * tn / (cm * cn > 1 ? 128.0 : (double)NUM_SMS));   // whole clusters per GPC
        const double t_comp = t_flop * (waves * NUM_SMS * (double)(TILE * TILE)) / ((double)M * (double)N);
        const double t_direct = std::max(t_link, t_comp) + 30e-6;
        if (direct_forced || !found || t_direct < best.t_model) {
            out->mb = M; out->nb = N; out->kb = Keff;
            out->h = out->w = out->kpanels = out->n_steps = 1;
            out->ksplit = 1;
            out->direct = 1;
            out->bytes_h2d = (uint64_t)rd; out->bytes_d2h = (uint64_t)wr;
            out->flops = scale_only ? 0.0 : 2.0 * (double)M * (double)N * (double)K;
            out->t_flop_s = t_flop; out->t_link_s = t_link; out->t_model_s = t_direct;
            return HCLOOC_OK;
        }
    }
    if (!found) return HCLOOC_ERR_BUDGET;
    out->mb = best.mb; out->nb = best.nb; out->kb = best.kb;
    out->h = best.h; out->w = best.w; out->kpanels = best.kpanels;
    out->n_steps = best.h * best.w * best.kpanels;
    out->n_sets = best.n_sets; out->n_abuf = best.n_abuf; out->n_bbuf = best.n_bbuf; out->ksplit = best.ksplit;
    out->lda_dev = best.lda_dev; out->ldb_dev = best.ldb_dev; out->ldc_dev = best.ldc_dev;
    out->bytes_a_buf = best.a_bytes; out->bytes_b_buf = best.b_bytes; out->bytes_c_buf = best.c_bytes;
    out->workspace_bytes = best.ws_bytes;
    out->c_on_device = c_dev ? (c_in_host ? 2 : 1) : 0;
    out->n_scratch = best.n_scratch; out->bytes_scratch = best.n_scratch ? streamk_scratch_bytes() : 0;
    out->bytes_h2d = best.bytes_h2d; out->bytes_d2h = best.bytes_d2h;
    out->n_copies_h2d = best.n_h2d; out->n_copies_d2h = best.n_d2h;
    out->flops = scale_only ? 0.0 : 2.0 * (double)M * (double)N * (double)K;
    out->t_flop_s = best.t_flop; out->t_link_s = best.t_link; out->t_model_s = best.t_model;
    return HCLOOC_OK;
}

extern "C" int hclooc_plan_trans(int64_t M, int64_t N, int64_t K, int beta_nonzero, int alpha_zero, size_t device_budget_bytes,
                                 int operands_on_device, int transa, int transb, hclooc_plan_t* out) {
    if (transa != HCL_OP_N && transa != HCL_OP_T) return -8;
    if (transb != HCL_OP_N && transb != HCL_OP_T) return -9;
    if (!out) return -10;
    return plan_impl(M, N, K, beta_nonzero, alpha_zero, device_budget_bytes, operands_on_device, transa, transb, out);
}

// The paper's rule, by divisor enumeration (example :301 -> (h, w) = (4, 2)).
extern "C" int hclMatrixPartitioner(int64_t M, int64_t N, int64_t K, int64_t budget_elements, int64_t* h, int64_t* w) {
    if (M <= 0) return -1;
    if (N <= 0) return -2;
    if (K <= 0) return -3;
    if (budget_elements <= 0) return -4;
    if (!h) return -5;
    if (!w) return -6;
    bool found = false;
    int64_t bh = 0, bw = 0;
    long double bt = 0;
    for (int64_t ww = 1; ww <= N; ++ww) {
        if (N % ww) continue;
        const int64_t nb = N / ww;
        // rows that fit beside one B slice: 2*mb*(K + nb) <= S - K*nb
        const long double left = (long double)budget_elements - (long double)K * nb;
        if (left <= 0) continue;
        const int64_t mb_max = (int64_t)std::floor(left / (2.0L * ((long double)K + nb)));
        if (mb_max < 1) continue;
        // traffic does not depend on h, so take the fewest row slices that fit (fewest steps)
        int64_t hh = ceil_div(M, std::min(M, mb_max));
        while (hh <= M && M % hh) ++hh;
        if (hh > M) continue;
        const long double traffic = (long double)ww * M * K + (long double)K * N + (long double)M * N;
        if (!found || traffic < bt || (traffic == bt && hh * ww < bh * bw) ||
            (traffic == bt && hh * ww == bh * bw && hh < bh)) {
            found = true; bt = traffic; bh = hh; bw = ww;
        }
    }
    if (!found) return HCLOOC_ERR_BUDGET;
    *h = bh; *w = bw;
    return HCLOOC_OK;
}

// Row bands for one process per GPU: independent C row blocks, no exchange step.
extern "C" int hclooc_shard_rows(int64_t M, int world, int rank, int64_t align, int64_t* row0, int64_t* rows) {
    if (M < 0) return -1;
    if (world < 1) return -2;
    if (rank < 0 || rank >= world) return -3;
    if (align < 1) return -4;
    if (!row0) return -5;
    if (!rows) return -6;
    const int64_t units = ceil_div(M, align);                  // bands are whole units of `align` rows
    const int64_t base = units / world, extra = units % world; // the first `extra` ranks get one unit more
    const int64_t u0 = rank * base + std::min<int64_t>(rank, extra);
    const int64_t un = base + (rank < extra ? 1 : 0);
    const int64_t r0 = std::min(M, u0 * align), r1 = std::min(M, (u0 + un) * align);
    *row0 = r0;
    *rows = r1 - r0;
    return HCLOOC_OK;
}
