// gtls_search: argument validation, device memory, the period-tile loop and the epilogue; and the
// two-stage search built on it.  All arithmetic of the search runs in the kernels; there is no CPU fallback.
#include <vector>

#include "api_common.cuh"

namespace gtls {
namespace api {

bool take_sort_scratch(Arena& ar, size_t tile, int n, SortScratch& sc) {
    const size_t nbk = (size_t)bucket_count_for(n), ncta = (size_t)bucket_cta_count(n);
    sc.hist = ar.take<unsigned short>(tile * ncta * nbk);
    sc.start = ar.take<u32>(tile * (nbk + 1));
    sc.rel = ar.take<u32>(tile * ncta * nbk);
    sc.fb_flag = ar.take<int>(tile);
    sc.fb_list = ar.take<int>(tile);
    sc.fb_count = ar.take<int>(1);
    return sc.fb_count != nullptr;
}

bool force_lsd_sort() {
    static const bool f = [] { const char* e = getenv("GTLS_SORT"); return e && strcmp(e, "lsd") == 0; }();
    return f;
}


// Steps a1-a4 for the tile described by `a` (a.perm, a.x1/s1[/x0/s0] are outputs).
//   The bucket fast path first; a period with a bucket larger than kBucketCap (clustered phases) is put
//   on the tile's fallback list on the device and skipped by the fast path; the LSD radix path
//   (fold_sort.cu + scan.cu) then runs over that list (a handful of CTAs that find it empty, normally).
//   GTLS_SORT=lsd: the LSD path for every period (A-B runs, tests).
// sort_only: permutation only.  phase_out: also export the phases (Eq. 10).
void run_fold_sort_scan(TileArgs& a, const SortScratch& sc, double* x2, double* s2, int pad_override,
                        bool sort_only, double* phase_out, cudaStream_t st, int* launches) {
    a.seg_list = nullptr; a.seg_count = nullptr;
    int nl = 0;
    if (!force_lsd_sort()) {
        BucketArgs b;
        memset(&b, 0, sizeof(b));
        b.n = a.n; b.tile = a.tile; b.p0 = a.p0; b.n_dur = a.n_dur; b.pad_override = pad_override;
        b.nbk = bucket_count_for(a.n);
        b.ncta = bucket_cta_count(a.n);
        int lg = 0; while ((1 << lg) < b.nbk) ++lg;
        b.shift = 32 - lg;
        b.pitch = a.pitch; b.spitch = a.spitch;
        b.t = a.t; b.wr = a.wr; b.w = a.w; b.wr2 = a.wr2; b.periods = a.periods; b.durtab = a.durtab;
        b.hist = sc.hist; b.start = sc.start; b.rel = sc.rel;
        b.fb_flag = sc.fb_flag; b.fb_list = sc.fb_list; b.fb_count = sc.fb_count;
        b.keys = a.keys_b; b.perm = a.perm;
        b.x1 = a.x1; b.s1 = a.s1; b.x0 = a.x0; b.s0 = a.s0; b.x2 = x2; b.s2 = s2;
        const bool has2 = s2 != nullptr, has0 = !a.uniform || has2;
        launch_bucket_sort_head(b, st);
        // the fallback list is known: the LSD path over it (a handful of CTAs, a few hundred microseconds
        // of latency when a period is on the list) runs beside the fast path on a side stream
        cudaStream_t ls = st;
        SideStream* side = side_stream(1);
        if (side) {
            cudaEventRecord(side->fork, st);
            cudaStreamWaitEvent(side->s, side->fork, 0);
            ls = side->s;
        }
        launch_bucket_sort_tail(b, has0, has2, sort_only, st);
        nl += sort_only ? 4 : 5;
        a.seg_list = sc.fb_list; a.seg_count = sc.fb_count;
        launch_fold_keys(a, nullptr, ls);
        int l2 = 0;
        const u64* sorted = launch_phase_sort(a, ls, &l2);
        if (!sort_only) launch_gather_scan(a, sorted, x2, s2, pad_override, ls);
        launch_perm_export(a, sorted, (int32_t*)a.perm, ls);
        if (side) {
            cudaEventRecord(side->join, ls);
            cudaStreamWaitEvent(st, side->join, 0);
        }
        if (phase_out) {                          // phases of every period: the LSD path's fold kernel, dense
            a.seg_list = nullptr; a.seg_count = nullptr;
            launch_fold_keys(a, phase_out, st); ++nl;
        }
        a.seg_list = nullptr; a.seg_count = nullptr;
        if (launches) *launches += nl + 1 + l2 + (sort_only ? 0 : 1) + 1;
        return;
    }
    launch_fold_keys(a, phase_out, st);
    int l2 = 0;
    const u64* sorted = launch_phase_sort(a, st, &l2);
    if (!sort_only) launch_gather_scan(a, sorted, x2, s2, pad_override, st);
    launch_perm_export(a, sorted, (int32_t*)a.perm, st);
    if (launches) *launches += nl + 1 + l2 + (sort_only ? 0 : 1) + 1;
}

}  // namespace api
}  // namespace gtls

using namespace gtls;
using namespace gtls::api;

// The search (gtls_search) and, with dbg_d / dbg_a set, its per-window debug export (gtls_ring_window_chi2: DEVICE
// arrays of ceil(n / stride) doubles for the ONE trial of a 1 period x 1 duration call on the general path).
static int search_impl(const double* t, const double* y, const double* dy, int64_t n,
                       const double* period_grid, int64_t n_per, const double* duration_grid,
                       int32_t n_dur, const double* tmpl, int32_t n_tmpl, const gtls_opts* opts,
                       double* out_chi2, gtls_best* out_best, double* out_sde_raw, double* out_sde,
                       gtls_summary* out_summary, double* dbg_d, double* dbg_a) {

    api::cuda_err_buf()[0] = 0;
    const gtls_opts o = resolve_opts(opts);
    if (!t || !y || !dy || !period_grid || !duration_grid || !tmpl || !out_chi2) return GTLS_EINVAL;
    if (n < 3 || n > 0x3fffffff || n_per < 1 || n_dur < 1 || n_dur > 4096 || n_tmpl < 2) return GTLS_EINVAL;
    if (!(o.dt0 >= 0.0) || o.sde_kernel < 0 || (o.sde_kernel > 1 && o.sde_kernel % 2 == 0)) return GTLS_EINVAL;
    if (o.path < 0 || o.path > 2 || o.period_tile < 0 || o.period_tile > 65535) return GTLS_EINVAL;   // (a tile is gridDim.y of the sort kernels)
    if (o.top_k < 0) return GTLS_EINVAL;
    if (o.top_k > kTopKMax || (o.top_k > 0 && o.chi2_fp32)) return GTLS_EUNSUPPORTED;
    if (o.chi2_fp32 != 0 && o.chi2_fp32 != 1) return GTLS_EINVAL;
    CU(cudaSetDevice(o.device));
    cudaStream_t st = (cudaStream_t)o.stream;
    const bool dev = o.pointers_on_device != 0;
    const long long n_durs_total = o.dur_per_period ? n_per * (long long)n_dur : n_dur;

    // ---- device memory -----------------------------------------------------------------
    Arena io;          // host mode: staged inputs and outputs
    if (!dev) {
        size_t bytes = 3 * align_up(n * 8) + align_up(n_per * 8) + align_up(n_durs_total * 8) +
                       align_up(n_tmpl * 8) + 3 * align_up(n_per * 8) +
                       align_up(n_per * sizeof(gtls_best)) + 16 * 256;
        int rc = alloc_arena(io, bytes);
        if (rc) return rc;
    }
    const double *d_t, *d_y, *d_dy, *d_per, *d_dur, *d_tmpl;
    int rc;
    if ((rc = stage_in(t, n, dev, io, st, &d_t))) return rc;
    if ((rc = stage_in(y, n, dev, io, st, &d_y))) return rc;
    if ((rc = stage_in(dy, n, dev, io, st, &d_dy))) return rc;
    if ((rc = stage_in(period_grid, n_per, dev, io, st, &d_per))) return rc;
    if ((rc = stage_in(duration_grid, n_durs_total, dev, io, st, &d_dur))) return rc;
    if ((rc = stage_in(tmpl, n_tmpl, dev, io, st, &d_tmpl))) return rc;
    double* d_chi2 = dev ? out_chi2 : io.take<double>(n_per);
    double* d_sde_raw_out = dev ? out_sde_raw : (out_sde_raw ? io.take<double>(n_per) : nullptr);
    double* d_sde_out = dev ? out_sde : (out_sde ? io.take<double>(n_per) : nullptr);
    gtls_best* d_best_out = dev ? out_best : (out_best ? io.take<gtls_best>(n_per) : nullptr);
    if (!d_chi2) return GTLS_ENOMEM;

    Arena ws;
    const Sizes worst = workspace_sizes(n, n_per, n_dur, 0.5, false);
    if (o.workspace) {
        ws.base = (char*)o.workspace; ws.size = o.workspace_bytes; ws.owned = false;
        if (((uintptr_t)ws.base & 255) != 0) return GTLS_EINVAL;
        if (ws.size < worst.fixed + align_up(worst.per_period)) return GTLS_ENOMEM;
    } else {
        // own scratch: the automatic tile, shrunk so that it takes at most half of the free device memory
        size_t need = gtls_workspace_bytes(n, n_per, n_dur, &o);
        size_t free_b = 0, total_b = 0;
        if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess && need > free_b / 2) {
            const size_t floor_b = worst.fixed + align_up(worst.per_period) + 64 * 256;
            need = free_b / 2 > floor_b ? free_b / 2 : floor_b;
        }
        if ((rc = alloc_arena(ws, need))) return rc;
    }
    double* d_wr = ws.take<double>(n);
    double* d_w = ws.take<double>(n);
    double* d_wr2 = ws.take<double>(n);
    CurveInfo* d_info = ws.take<CurveInfo>(1);
    SdeScratch* d_sde_sc = ws.take<SdeScratch>(1);
    unsigned long long* d_counters = ws.take<unsigned long long>(2);
    double* d_sde_raw = d_sde_raw_out ? d_sde_raw_out : ws.take<double>(n_per);
    double* d_sde = d_sde_out ? d_sde_out : ws.take<double>(n_per);
    gtls_best* d_best = d_best_out ? d_best_out : ws.take<gtls_best>(n_per);
    if (!d_best) return GTLS_ENOMEM;

    Timer tm;
    tm.init(o.stats != nullptr, st);
    tm.mark(9);                                   // begin of the call (events 9 / 10 belong to the Timer: no leak on early returns)
    gtls_stats stats;
    memset(&stats, 0, sizeof(stats));

    // ---- a0: per-curve arrays + validation ----------------------------------------------
    tm.mark(0);
    CU(cudaMemsetAsync(d_info, 0, sizeof(CurveInfo), st));
    CU(cudaMemsetAsync(d_counters, 0, 2 * sizeof(unsigned long long), st));
    launch_curve_pre(d_t, d_y, d_dy, (int)n, d_wr, d_w, d_wr2, d_info, st);
    launch_grid_check(d_per, n_per, d_dur, n_durs_total, d_info, st);
    stats.kernel_launches += 2;
    CurveInfo info;
    CU(cudaMemcpyAsync(&info, d_info, sizeof(info), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    CU(cudaGetLastError());
    if (info.bad_curve) return GTLS_ENONFINITE;
    if (info.bad_period || info.bad_duration) return GTLS_EGRID;
    tm.mark(1);
    if (o.stats) { CU(cudaStreamSynchronize(st)); stats.ms_pre += tm.ms(0, 1); }
    const bool uniform = info.w_min == info.w_max;

    const double* gtab_dev = nullptr;
    int gtab_max = 0;
    {   // template sums per D, once per search (every D the grid can ask for: D <= floor(q_max * n) <= pitch - n)
        long long dmax = (long long)(info.q_max * (double)n);
        dmax = dmax < 1 ? 1 : (dmax > n - 1 ? n - 1 : dmax);
        double* gtab = ws.take<double>(2 * (size_t)(dmax + 1));
        if (!gtab) return GTLS_ENOMEM;
        launch_gtab(d_tmpl, n_tmpl, (int)dmax, gtab, st);
        stats.kernel_launches += 1;
        gtab_dev = gtab; gtab_max = (int)dmax;
    }

    // ---- path: fused small-N kernel (small.cu) when the folded curve fits a CTA's shared memory -------
    // opts->path: 0 automatic, 1 force the fused path (GTLS_EUNSUPPORTED when it does not apply), 2 force
    // the general tiled path
    const bool small_ok = uniform && o.top_k == 0 && o.chi2_fp32 == 0 && n <= 65535 &&
                          small_path_fits((int)n, gtab_max, n_dur, o.dt0);
    if (o.path == 1 && !small_ok) return GTLS_EUNSUPPORTED;
    const bool use_small = small_ok && o.path != 2 && (!dbg_d || o.path == 1);   // (the debug export names its path)
    int tile = 0;
    SdeScratch sc;
    unsigned long long counters[2];
    if (use_small) {
        long long* d_off = ws.take<long long>(4);                 // curve_off[2], per_off[2]
        unsigned long long* d_queue = ws.take<unsigned long long>(1);
        if (!d_queue) return GTLS_ENOMEM;
        const long long h_off[4] = {0, (long long)n, 0, (long long)n_per};
        CU(cudaMemcpyAsync(d_off, h_off, sizeof(h_off), cudaMemcpyHostToDevice, st));
        CU(cudaMemsetAsync(d_queue, 0, sizeof(unsigned long long), st));
        SmallArgs sa;
        memset(&sa, 0, sizeof(sa));
        sa.n_items = n_per; sa.n_dur = n_dur; sa.n_tmpl = n_tmpl; sa.dur_per_period = o.dur_per_period; sa.dt0 = o.dt0;
        sa.curve_off = d_off; sa.per_off = d_off + 2;
        sa.t = d_t; sa.wr = d_wr; sa.info = d_info; sa.periods = d_per; sa.durs = d_dur; sa.tmpl = d_tmpl;
        sa.gtab = gtab_dev; sa.out_chi2 = d_chi2; sa.out_best = d_best; sa.counters = d_counters; sa.queue = d_queue;
        sa.dbg_dchi2 = dbg_d; sa.dbg_depth = dbg_a;
        int sms = 0;
        CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, o.device));
        tm.mark(4);
        const int ce = launch_tls_small(sa, (int)n, gtab_max, sms, st);
        if (ce != 0) return cuda_fail((cudaError_t)ce, "k_tls_small");
        tm.mark(5);
        stats.kernel_launches += 1;
        stats.chi2_launches += 1;
        if (o.stats) { CU(cudaStreamSynchronize(st)); stats.ms_chi2 += tm.ms(4, 5); }
    } else {
        // ---- tile geometry -------------------------------------------------------------------
        const Sizes sz = workspace_sizes(n, n_per, n_dur, info.q_max, uniform);
        const size_t avail = ws.size - align_up(ws.off) - 32 * 256;
        long long tile_cap = (long long)(avail / align_up(sz.per_period + 8 * 256));
        tile = o.period_tile > 0 ? o.period_tile : auto_tile(n_per, sz, kDefaultTileBudget);
        if (tile > tile_cap) tile = (int)tile_cap;
        if (o.period_tile <= 0 && tile >= kFinishSlots && tile < n_per) tile -= (int)(tile % kFinishSlots);   // see auto_tile
        if (tile > n_per) tile = (int)n_per;
        if (tile < 1) return GTLS_ENOMEM;
        TileArgs a;
        memset(&a, 0, sizeof(a));
        a.n = (int)n; a.n_dur = n_dur; a.n_tmpl = n_tmpl; a.dur_per_period = o.dur_per_period;
        a.dt0 = o.dt0; a.uniform = uniform ? 1 : 0; a.w_uniform = info.w_min; a.chi2_fp32 = o.chi2_fp32; a.top_k = o.top_k;
        a.pitch = pitch_for(n, info.q_max); a.spitch = a.pitch + 8;
        a.t = d_t; a.wr = d_wr; a.w = d_w; a.wr2 = d_wr2; a.periods = d_per; a.durs = d_dur;
        a.tmpl = d_tmpl; a.chi2_0 = &d_info->chi2_0;
        a.dbg_dchi2 = dbg_d; a.dbg_depth = dbg_a;
        const int nt = (int)((n + kRadixTile - 1) / kRadixTile);
        a.keys_a = ws.take<u64>((size_t)tile * n);
        a.keys_b = ws.take<u64>((size_t)tile * n);
        a.counts = ws.take<u32>((size_t)tile * 256 * nt);
        a.perm = ws.take<u32>((size_t)tile * n);
        SortScratch ssc;
        if (!take_sort_scratch(ws, (size_t)tile, (int)n, ssc)) return GTLS_ENOMEM;
        a.durtab = ws.take<DurEntry>((size_t)tile * n_dur);
        a.gtab = gtab_dev; a.gtab_max = gtab_max;
        a.partial = ws.take<Partial>((size_t)tile * n_dur);
        a.trial_list = ws.take<int>((size_t)kChi2Variants * tile * n_dur);
        a.trial_count = ws.take<int>((size_t)kChi2Variants * (2 + kBinBlocks));   // totals, the per-CTA counts of k_bin_trials, the trial queues
        a.x1 = ws.take<double>((size_t)tile * a.pitch + kXMargin);      // + the last period's zero margin
        a.s1 = ws.take<double>((size_t)tile * a.spitch);
        if (!uniform) {
            a.x0 = ws.take<double>((size_t)tile * a.pitch + kXMargin);
            a.s0 = ws.take<double>((size_t)tile * a.spitch);
        }
        if (!a.s1 || (!uniform && !a.s0)) return GTLS_ENOMEM;

        // ---- period tiles ----------------------------------------------------------------------
        for (long long p0 = 0; p0 < n_per; p0 += tile) {
            a.p0 = p0;
            a.tile = (int)((n_per - p0) < tile ? (n_per - p0) : tile);
            int launches = 0;
            tm.mark(0);
            launch_durtab(a, st);
            tm.mark(1);
            tm.mark(2);
            run_fold_sort_scan(a, ssc, nullptr, nullptr, -1, false, nullptr, st, &launches);
            tm.mark(3);
            tm.mark(4);
            if (a.top_k > 0) launch_chi2_topk(a, st);
            else launch_chi2_ring(a, st);
            tm.mark(5);
            launch_reduce(a, d_chi2, d_best, d_counters, st);
            tm.mark(6);
            stats.kernel_launches += launches + 2 + (a.top_k > 0 ? 1 : 2 + (uniform ? kChi2Variants - 1 : kChi2Variants - 3));   // k_bin_trials is two launches
            stats.chi2_launches += 1;
            if (o.stats) {
                CU(cudaStreamSynchronize(st));
                stats.ms_pre += tm.ms(0, 1); stats.ms_fold += tm.ms(1, 2); stats.ms_sort += tm.ms(2, 3);
                stats.ms_scan += tm.ms(3, 4); stats.ms_chi2 += tm.ms(4, 5); stats.ms_reduce += tm.ms(5, 6);
            }
        }
    }
    CU(cudaGetLastError());

    // ---- a9: SR / SDE epilogue --------------------------------------------------------------
    tm.mark(0);
    int launches = 0;
    launch_sde(d_chi2, n_per, o.sde_kernel, d_sde_raw, d_sde, d_sde_sc, st, &launches);
    stats.kernel_launches += launches;
    tm.mark(1);
    CU(cudaMemcpyAsync(&sc, d_sde_sc, sizeof(sc), cudaMemcpyDeviceToHost, st));
    CU(cudaMemcpyAsync(counters, d_counters, sizeof(counters), cudaMemcpyDeviceToHost, st));
    tm.mark(10);
    CU(cudaStreamSynchronize(st));
    CU(cudaGetLastError());
    if (o.stats) stats.ms_epilogue = tm.ms(0, 1);

    if (out_summary) {
        gtls_best b;
        double period = 0.0;
        CU(cudaMemcpyAsync(&b, d_best + sc.argmin, sizeof(b), cudaMemcpyDeviceToHost, st));
        CU(cudaMemcpyAsync(&period, d_per + sc.argmin, sizeof(double), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        out_summary->best_period_idx = sc.argmin;
        out_summary->best_dur_idx = b.dur_idx;
        out_summary->best_start = b.start;
        out_summary->best_period = period;
        out_summary->best_t0 = b.t0;
        out_summary->best_depth = b.depth;
        out_summary->chi2_min = sc.chi2_min;
        out_summary->chi2_null = info.chi2_0;
        out_summary->sde_raw_max = sc.sde_raw_best;
        out_summary->sde_max = sc.sde_max;
        out_summary->sde_argmax = sc.sde_argmax;
        out_summary->windows_evaluated = (int64_t)counters[0];
    }
    if (!dev) {
        CU(cudaMemcpyAsync(out_chi2, d_chi2, n_per * sizeof(double), cudaMemcpyDeviceToHost, st));
        if (out_best) CU(cudaMemcpyAsync(out_best, d_best, n_per * sizeof(gtls_best), cudaMemcpyDeviceToHost, st));
        if (out_sde_raw) CU(cudaMemcpyAsync(out_sde_raw, d_sde_raw, n_per * sizeof(double), cudaMemcpyDeviceToHost, st));
        if (out_sde) CU(cudaMemcpyAsync(out_sde, d_sde, n_per * sizeof(double), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
    }
    if (o.stats) {
        stats.ms_total = tm.ms(9, 10);
        stats.windows = (int64_t)counters[0];
        stats.window_points = (int64_t)counters[1];
        stats.period_points = n * n_per;
        stats.period_tile = tile;
        stats.path = use_small ? 1 : 2;
        stats.uniform_dy = uniform ? 1 : 0;
        *o.stats = stats;
    }
    io.idle = ws.idle = true;                 // the stream was synchronised after the last use of both
    return sc.degenerate ? GTLS_EDEGENERATE : GTLS_OK;
}


extern "C" {

size_t gtls_workspace_bytes(int64_t n, int64_t n_per, int32_t n_dur, const gtls_opts* opts) {
    if (n < 3 || n_per < 1 || n_dur < 1) return 0;
    const gtls_opts o = resolve_opts(opts);
    const Sizes s = workspace_sizes(n, n_per, n_dur, 0.5, false);     // worst case
    const int tile = o.period_tile > 0 ? (int)(o.period_tile < n_per ? o.period_tile : n_per)
                                       : auto_tile(n_per, s, kDefaultTileBudget);
    size_t bytes = s.fixed + (size_t)tile * align_up(s.per_period) + 64 * 256;
    if (o.period_tile <= 0) {
        // ... and enough for the common case (one common error bar, durations up to a fifth of the period) to run at
        // ITS automatic tile, which is larger than the worst case's (c4: 4144 periods against 2368)
        const Sizes c = workspace_sizes(n, n_per, n_dur, 0.2, true);
        const size_t common = s.fixed + (size_t)auto_tile(n_per, c, kDefaultTileBudget) * align_up(c.per_period + 8 * 256) + 64 * 256;
        if (common > bytes) bytes = common;
    }
    return bytes;
}

int gtls_search(const double* t, const double* y, const double* dy, int64_t n,
                const double* period_grid, int64_t n_per, const double* duration_grid,
                int32_t n_dur, const double* tmpl, int32_t n_tmpl, const gtls_opts* opts,
                double* out_chi2, gtls_best* out_best, double* out_sde_raw, double* out_sde,
                gtls_summary* out_summary) {
    return search_impl(t, y, dy, n, period_grid, n_per, duration_grid, n_dur, tmpl, n_tmpl, opts, out_chi2, out_best,
                       out_sde_raw, out_sde, out_summary, nullptr, nullptr);
}

int64_t gtls_ring_window_chi2(const double* t, const double* y, const double* dy, int64_t n, double period,
                              double q, const double* tmpl, int32_t n_tmpl, const gtls_opts* opts,
                              int32_t* out_start, double* out_depth, double* out_dchi2, double* out_chi2_null) {
    cuda_err_buf()[0] = 0;
    gtls_opts o = resolve_opts(opts);
    if (!t || !y || !dy || !tmpl || !out_start || !out_depth || !out_dchi2) return GTLS_EINVAL;
    if (n < 3 || n > 0x3fffffff || n_tmpl < 2 || !(period > 0.0) || !(q > 0.0) || !(q <= 0.5) || !(o.dt0 >= 0.0)) return GTLS_EINVAL;
    if (o.pointers_on_device) return GTLS_EUNSUPPORTED;          // a host-pointer debug export
    if (o.top_k != 0 || o.chi2_fp32 != 0) return GTLS_EUNSUPPORTED;
    CU(cudaSetDevice(o.device));
    cudaStream_t st = (cudaStream_t)o.stream;
    long long D = (long long)(q * (double)n);
    D = D < 1 ? 1 : (D > n - 1 ? n - 1 : D);
    long long stride = o.dt0 > 0.0 ? (long long)((double)D * o.dt0) : 1;
    if (stride < 1) stride = 1;
    const long long nW = (n + stride - 1) / stride;
    Arena ar;
    int rc = alloc_arena(ar, 2 * align_up(nW * 8) + 1024);
    if (rc) return rc;
    double* d_d = ar.take<double>(nW);
    double* d_a = ar.take<double>(nW);
    if (!d_a) return GTLS_ENOMEM;
    CU(cudaMemsetAsync(d_d, 0xff, nW * 8, st));                   // NaN: a window the kernel did not score stays visible
    CU(cudaMemsetAsync(d_a, 0xff, nW * 8, st));
    o.path = o.path == 1 ? 1 : 2;          // 1: the fused small-N kernel (GTLS_EUNSUPPORTED where it does not apply)
    o.sde_kernel = 0; o.period_tile = 0; o.dur_per_period = 0; o.stats = nullptr;
    o.workspace = nullptr; o.workspace_bytes = 0;
    double chi2 = 0.0;
    gtls_summary summ;
    memset(&summ, 0, sizeof(summ));
    rc = search_impl(t, y, dy, n, &period, 1, &q, 1, tmpl, n_tmpl, &o, &chi2, nullptr, nullptr, nullptr, &summ, d_d, d_a);
    if (rc != GTLS_OK && rc != GTLS_EDEGENERATE) return rc;
    CU(cudaMemcpyAsync(out_dchi2, d_d, nW * 8, cudaMemcpyDeviceToHost, st));
    CU(cudaMemcpyAsync(out_depth, d_a, nW * 8, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    ar.idle = true;
    for (long long k = 0; k < nW; ++k) out_start[k] = (int32_t)(k * stride);
    if (out_chi2_null) *out_chi2_null = summ.chi2_null;
    return nW;
}

int gtls_search_two_stage(const double* t, const double* y, const double* dy, int64_t n,
                          const double* period_grid, int64_t n_per, const double* duration_grid,
                          int32_t n_dur, const double* tmpl, int32_t n_tmpl, const gtls_opts* opts,
                          int32_t n_refine, double* out_chi2, gtls_best* out_best, double* out_sde_raw,
                          double* out_sde, int64_t* out_refined, gtls_summary* out_summary) {
    api::cuda_err_buf()[0] = 0;
    const gtls_opts o = resolve_opts(opts);
    if (!t || !y || !dy || !period_grid || !duration_grid || !tmpl || !out_chi2 || !out_best) return GTLS_EINVAL;
    if (n < 3 || n_per < 1 || n_dur < 1 || n_tmpl < 2 || n_refine <= 0) return GTLS_EINVAL;
    CU(cudaSetDevice(o.device));
    cudaStream_t st = (cudaStream_t)o.stream;
    const bool dev = o.pointers_on_device != 0;
    const long long n_durs_total = o.dur_per_period ? n_per * (long long)n_dur : n_dur;
    const int K = (int)(n_refine < n_per ? n_refine : n_per);

    // device copies of everything (host mode), and the stage-2 scratch
    Arena ar;
    size_t bytes = align_up(n_per) + align_up((size_t)K * 8) * 3 + align_up((size_t)K * n_dur * 8) +
                   align_up((size_t)K * sizeof(gtls_best)) + 2 * align_up(n_per * 8) + 32 * 256;
    if (!dev)
        bytes += 3 * align_up(n * 8) + align_up(n_per * 8) + align_up(n_durs_total * 8) + align_up(n_tmpl * 8) +
                 align_up(n_per * 8) + align_up(n_per * sizeof(gtls_best));
    int rc = alloc_arena(ar, bytes);
    if (rc) return rc;
    const double *d_t, *d_y, *d_dy, *d_per, *d_dur, *d_tmpl;
    if ((rc = stage_in(t, n, dev, ar, st, &d_t))) return rc;
    if ((rc = stage_in(y, n, dev, ar, st, &d_y))) return rc;
    if ((rc = stage_in(dy, n, dev, ar, st, &d_dy))) return rc;
    if ((rc = stage_in(period_grid, n_per, dev, ar, st, &d_per))) return rc;
    if ((rc = stage_in(duration_grid, n_durs_total, dev, ar, st, &d_dur))) return rc;
    if ((rc = stage_in(tmpl, n_tmpl, dev, ar, st, &d_tmpl))) return rc;
    double* d_chi2 = dev ? out_chi2 : ar.take<double>(n_per);
    gtls_best* d_best = dev ? out_best : ar.take<gtls_best>(n_per);
    double* d_sde_raw = (dev && out_sde_raw) ? out_sde_raw : ar.take<double>(n_per);
    double* d_sde = (dev && out_sde) ? out_sde : ar.take<double>(n_per);
    unsigned char* d_mark = ar.take<unsigned char>(n_per);
    long long* d_sel = ar.take<long long>(K);
    double* d_per2 = ar.take<double>(K);
    double* d_dur2 = ar.take<double>((size_t)K * n_dur);
    double* d_chi2b = ar.take<double>(K);
    gtls_best* d_bestb = ar.take<gtls_best>(K);
    if (!d_bestb) return GTLS_ENOMEM;

    // ---- stage 1: coarse search over all periods ---------------------------------------------------
    gtls_opts o1 = o;
    o1.pointers_on_device = 1;
    o1.stats = nullptr;
    gtls_summary s1, s2, s3;
    memset(&s1, 0, sizeof(s1)); memset(&s2, 0, sizeof(s2)); memset(&s3, 0, sizeof(s3));
    rc = gtls_search(d_t, d_y, d_dy, n, d_per, n_per, d_dur, n_dur, d_tmpl, n_tmpl, &o1, d_chi2, d_best,
                     d_sde_raw, d_sde, &s1);
    int rc_final = rc;
    const bool refined = rc == GTLS_OK;
    if (refined) {
        // ---- stage 2: the K periods of highest SDE, every trial T0 -------------------------------------
        launch_topk_sde(d_sde, n_per, K, d_mark, d_sel, st);
        launch_gather_refine(d_per, d_dur, o.dur_per_period, n_dur, d_sel, K, d_per2, d_dur2, st);
        gtls_opts o2 = o1;
        o2.dt0 = 0.0;
        o2.dur_per_period = 1;
        o2.sde_kernel = 0;
        rc = gtls_search(d_t, d_y, d_dy, n, d_per2, K, d_dur2, n_dur, d_tmpl, n_tmpl, &o2, d_chi2b, d_bestb,
                         nullptr, nullptr, &s2);
        if (rc != GTLS_OK && rc != GTLS_EDEGENERATE) return rc;
        launch_merge_refined(d_sel, K, d_chi2b, d_bestb, d_chi2, d_best, st);
        rc_final = gtls_sde(d_chi2, n_per, &o1, d_sde_raw, d_sde, &s3);
        if (rc_final != GTLS_OK && rc_final != GTLS_EDEGENERATE) return rc_final;
    } else if (rc != GTLS_EDEGENERATE) {
        return rc;
    }
    if (out_summary) {
        *out_summary = s1;
        if (refined) {
            out_summary->best_period_idx = s3.best_period_idx;
            out_summary->chi2_min = s3.chi2_min;
            out_summary->sde_raw_max = s3.sde_raw_max;
            out_summary->sde_max = s3.sde_max;
            out_summary->sde_argmax = s3.sde_argmax;
            gtls_best b;
            double period = 0.0;
            CU(cudaMemcpyAsync(&b, d_best + s3.best_period_idx, sizeof(b), cudaMemcpyDeviceToHost, st));
            CU(cudaMemcpyAsync(&period, d_per + s3.best_period_idx, sizeof(double), cudaMemcpyDeviceToHost, st));
            CU(cudaStreamSynchronize(st));
            out_summary->best_dur_idx = b.dur_idx; out_summary->best_start = b.start;
            out_summary->best_period = period; out_summary->best_t0 = b.t0; out_summary->best_depth = b.depth;
        }
        out_summary->windows_evaluated = s1.windows_evaluated + s2.windows_evaluated;
    }
    const cudaMemcpyKind d2x = dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    if (out_refined && refined)
        CU(cudaMemcpyAsync(out_refined, d_sel, (size_t)K * sizeof(long long), d2x, st));
    if (!dev) {
        CU(cudaMemcpyAsync(out_chi2, d_chi2, n_per * sizeof(double), cudaMemcpyDeviceToHost, st));
        CU(cudaMemcpyAsync(out_best, d_best, n_per * sizeof(gtls_best), cudaMemcpyDeviceToHost, st));
        if (out_sde_raw) CU(cudaMemcpyAsync(out_sde_raw, d_sde_raw, n_per * sizeof(double), cudaMemcpyDeviceToHost, st));
        if (out_sde) CU(cudaMemcpyAsync(out_sde, d_sde, n_per * sizeof(double), cudaMemcpyDeviceToHost, st));
    }
    CU(cudaStreamSynchronize(st));
    CU(cudaGetLastError());
    return rc_final;
}

}  // extern "C"
