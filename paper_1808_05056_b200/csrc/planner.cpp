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
constexpr double OVERLAP_PENALTY = 0.10;
}  // namespace

const MachineModel& machine_model() {
    static const MachineModel mm = {
        env_or("HCLOOC_FP64_TFLOPS", 37.17) * 1e12,   // DMMA loop, 148 SMs, sustained (profiles/r01_box_probe.md)
        env_or("HCLOOC_H2D_GBPS", 55.5) * 1e9,
        env_or("HCLOOC_D2H_GBPS", 51.5) * 1e9,
        env_or("HCLOOC_DUPLEX_GBPS", 88.0) * 1e9,
        env_or("HCLOOC_COPY_LATENCY_US", 4.0) * 1e-6,
        env_or("HCLOOC_LAUNCH_LATENCY_US", 5.0) * 1e-6,
    };
    return mm;
}

namespace {

struct Cand {
    int64_t mb, nb, kb, h, w, kpanels;
    int n_sets, n_bbuf, ksplit;
    int64_t lda_dev, ldb_dev, ldc_dev;
    uint64_t a_bytes, b_bytes, c_bytes, ws_bytes;
    uint64_t bytes_h2d, bytes_d2h, n_h2d, n_d2h;
    double t_flop, t_link, t_model;
};

// Number of chunks the executor splits a prefetched B slice into (one per step of the previous
// column, so the prefetch interleaves with that column's A/C uploads).
int64_t prefetch_chunks(int64_t h, int64_t kk) { return std::max<int64_t>(1, std::min(h, kk)); }

void fill_traffic(Cand& c, int64_t M, int64_t N, int64_t K, bool beta_nz, bool scale_only) {
    const uint64_t MN = (uint64_t)M * (uint64_t)N;
    const uint64_t steps = (uint64_t)c.h * c.w * c.kpanels;
    const bool cload0 = beta_nz;
    uint64_t el_h2d = 0, n_h2d = 0;
    if (!scale_only) {
        el_h2d += (uint64_t)c.w * (uint64_t)M * (uint64_t)K;       // every A slice once per column of blocks
        el_h2d += (uint64_t)K * (uint64_t)N;                       // every B slice once
        n_h2d += steps;                                            // one A copy per step
        const uint64_t slabs = (uint64_t)c.w * c.kpanels;
        if (c.n_bbuf == 1) n_h2d += slabs;
        else {
            n_h2d += 1;                                            // first slice in one piece
            for (int64_t p = 0; p < c.kpanels; ++p) {
                const int64_t kk = std::min(c.kb, K - p * c.kb);
                n_h2d += (uint64_t)c.w * prefetch_chunks(c.h, kk);
            }
            n_h2d -= prefetch_chunks(c.h, std::min(c.kb, K));      // slice 0 was counted as chunks too
        }
    }
    if (cload0) { el_h2d += MN; n_h2d += (uint64_t)c.h * c.w; }
    if (c.kpanels > 1) { el_h2d += (uint64_t)(c.kpanels - 1) * MN; n_h2d += (uint64_t)(c.kpanels - 1) * c.h * c.w; }
    c.bytes_h2d = 8 * el_h2d;
    c.n_h2d = n_h2d;
    c.bytes_d2h = 8 * (uint64_t)c.kpanels * MN;
    c.n_d2h = steps;
}

void cost(Cand& c, int64_t M, int64_t N, int64_t K, bool beta_nz, bool scale_only) {
    const MachineModel& mm = machine_model();
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
    // too few tiles in flight to fill the SMs: a cluster of 2 or 4 CTAs shares each tile's K range
    const int force_ks = (int)env_or("HCLOOC_FORCE_KSPLIT", 0);
    c.ksplit = scale_only ? 1 : (force_ks ? force_ks : dgemm_auto_ksplit((int64_t)(std::max(1, c.n_sets - 2) * tiles_step), c.kb));
    const double in_flight = std::max(1, c.n_sets - 2) * tiles_step * c.ksplit;
    double fill = std::min(1.0, in_flight / NUM_SMS);
    if (tiles_step >= NUM_SMS) fill = std::min(fill, 0.98);
    c.t_flop = flops / mm.fp64_flops;
    const double t_compute = c.t_flop / std::max(1e-3, pad_eff * fill) + steps * 1e-6;
    const double t_in = c.bytes_h2d / mm.h2d_Bps + c.n_h2d * mm.copy_latency_s;
    const double t_out = c.bytes_d2h / mm.d2h_Bps + c.n_d2h * mm.copy_latency_s;
    c.t_link = std::max(std::max(t_in, t_out), (double)(c.bytes_h2d + c.bytes_d2h) / mm.duplex_Bps);
    const bool cload = beta_nz || c.kpanels > 1;
    const double t_pro = ((double)c.b_bytes + (double)c.a_bytes + (cload ? (double)c.c_bytes : 0.0)) / mm.h2d_Bps + 3 * mm.copy_latency_s;
    const double t_step = t_compute / std::max(1.0, steps);
    const double switches = (double)c.w * c.kpanels - 1.0;
    double comp_path = t_pro + t_compute;
    double link_path = c.t_link;
    if (c.n_bbuf == 1) {
        comp_path += switches * ((double)c.b_bytes / mm.h2d_Bps);   // compute idles while the next B slice loads
        link_path += switches * t_step * std::min<double>(c.n_sets, 3);  // link idles while the column drains
    }
    const double t_tail = t_step * std::max(1.0, tiles_step / NUM_SMS > 1 ? 1.0 : 1.0) + (double)c.c_bytes / mm.d2h_Bps + mm.copy_latency_s;
    // imperfect overlap: the shorter path still costs a fraction of its length (bursty uploads, shared
    // DMA/HBM resources), which also keeps plans away from the edge where link time ~ compute time
    c.t_model = std::max(comp_path, link_path) + OVERLAP_PENALTY * std::min(comp_path, link_path) + t_tail + mm.launch_latency_s;
}

}  // namespace
}  // namespace hclooc

using namespace hclooc;

extern "C" int hclooc_plan(int64_t M, int64_t N, int64_t K, int beta_nonzero, int alpha_zero,
                           size_t device_budget_bytes, hclooc_plan_t* out) {
    if (M < 0) return -1;
    if (N < 0) return -2;
    if (K < 0) return -3;
    if (!out) return -7;
    std::memset(out, 0, sizeof(*out));
    out->M = M; out->N = N; out->K = K;
    out->beta_nonzero = beta_nonzero ? 1 : 0;
    const bool scale_only = (alpha_zero != 0) || (K == 0);
    out->scale_only = scale_only ? 1 : 0;
    if (M == 0 || N == 0) return HCLOOC_OK;                       // nothing to do: zero steps
    const bool beta_nz = beta_nonzero != 0;
    const int64_t Keff = scale_only ? 0 : K;
    const uint64_t S = (uint64_t)device_budget_bytes;

    // experiment knobs (not part of the ABI): force parts of the plan
    const int64_t force_nb = (int64_t)env_or("HCLOOC_FORCE_NB", 0), force_mb = (int64_t)env_or("HCLOOC_FORCE_MB", 0);
    const int force_sets = (int)env_or("HCLOOC_FORCE_SETS", 0), force_bbuf = (int)env_or("HCLOOC_FORCE_BBUF", 0);
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
            const int64_t lda_dev = round_up(std::max<int64_t>(kb, 1), LD_ALIGN);
            const int64_t ldb_dev = round_up(nb, LD_ALIGN), ldc_dev = ldb_dev;
            const uint64_t b_bytes = scale_only ? 0 : round_up((uint64_t)kb * ldb_dev * 8, BUF_ALIGN);
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
                    if (top >= TILE) top = top / TILE * TILE; else if (top >= 8) top = top / 8 * 8;
                    tried[nt++] = top;
                    for (int64_t cand_mb : {(int64_t)1024, (int64_t)512, (int64_t)256, (int64_t)128})
                        if (cand_mb < top) tried[nt++] = cand_mb;
                    if (force_mb) { nt = 0; if (force_mb <= std::min(M, rows_max)) tried[nt++] = force_mb; }
                    for (int q = 0; q < nt; ++q) {
                        Cand c{};
                        c.mb = tried[q]; c.nb = nb; c.kb = kb; c.kpanels = kp;
                        c.h = ceil_div(M, c.mb); c.w = weff;
                        c.n_sets = (int)std::min<int64_t>(n_sets, std::max<int64_t>(2, c.h * c.w * kp));
                        c.n_bbuf = n_bbuf;
                        c.lda_dev = scale_only ? 0 : lda_dev; c.ldb_dev = scale_only ? 0 : ldb_dev; c.ldc_dev = ldc_dev;
                        c.a_bytes = scale_only ? 0 : round_up((uint64_t)c.mb * lda_dev * 8, BUF_ALIGN);
                        c.b_bytes = b_bytes;
                        c.c_bytes = round_up((uint64_t)c.mb * ldc_dev * 8, BUF_ALIGN);
                        c.ws_bytes = (uint64_t)n_bbuf * b_bytes + (uint64_t)c.n_sets * (c.a_bytes + c.c_bytes);
                        if (c.ws_bytes > S) continue;
                        cost(c, M, N, Keff, beta_nz, scale_only);
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
    if (!found) return HCLOOC_ERR_BUDGET;
    out->mb = best.mb; out->nb = best.nb; out->kb = best.kb;
    out->h = best.h; out->w = best.w; out->kpanels = best.kpanels;
    out->n_steps = best.h * best.w * best.kpanels;
    out->n_sets = best.n_sets; out->n_bbuf = best.n_bbuf; out->ksplit = best.ksplit;
    out->lda_dev = best.lda_dev; out->ldb_dev = best.ldb_dev; out->ldc_dev = best.ldc_dev;
    out->bytes_a_buf = best.a_bytes; out->bytes_b_buf = best.b_bytes; out->bytes_c_buf = best.c_bytes;
    out->workspace_bytes = best.ws_bytes;
    out->bytes_h2d = best.bytes_h2d; out->bytes_d2h = best.bytes_d2h;
    out->n_copies_h2d = best.n_h2d; out->n_copies_d2h = best.n_d2h;
    out->flops = scale_only ? 0.0 : 2.0 * (double)M * (double)N * (double)K;
    out->t_flop_s = best.t_flop; out->t_link_s = best.t_link; out->t_model_s = best.t_model;
    return HCLOOC_OK;
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
