// dd_api.cu -- the C ABI of include/dd.h: argument checking, table upload, kernel launch.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "dd_kernels.cuh"
#include "dd_plan.h"

namespace dd {

static thread_local std::string g_cuda_error;

static dd_status cuda_fail(cudaError_t e, const char *what)
{
    g_cuda_error = std::string(what) + ": " + cudaGetErrorName(e) + " (" + cudaGetErrorString(e) + ")";
    (void)cudaGetLastError();   // clear the sticky-less error state
    return DD_ERR_CUDA;
}

// for the other files of the library that return statuses (dd_tree.cu)
dd_status report_cuda_error(cudaError_t e, const char *what) { return cuda_fail(e, what); }
void set_error_text(const std::string &text) { g_cuda_error = text; }

// Device staging of dd_execute_host: the whole packed input plus two output slabs.
struct HostStage {
    uint8_t *d_in = nullptr;
    size_t in_bytes = 0;
    uint8_t *d_out[2] = {nullptr, nullptr};
    size_t out_bytes = 0;
    cudaStream_t copy_in = nullptr, compute = nullptr, copy_out[2] = {nullptr, nullptr};
    cudaEvent_t in_ready = nullptr, in_rest = nullptr, done[2] = {nullptr, nullptr}, drained[2] = {nullptr, nullptr};
    bool streams = false;
};

static void free_stage(HostStage *s)
{
    if (!s)
        return;
    cudaFree(s->d_in);
    cudaFree(s->d_out[0]);
    cudaFree(s->d_out[1]);
    if (s->streams) {
        cudaStreamDestroy(s->copy_in);
        cudaStreamDestroy(s->compute);
        for (int i = 0; i < 2; ++i) {
            cudaStreamDestroy(s->copy_out[i]);
            cudaEventDestroy(s->done[i]);
            cudaEventDestroy(s->drained[i]);
        }
        cudaEventDestroy(s->in_ready);
        if (s->in_rest)
            cudaEventDestroy(s->in_rest);
    }
    delete s;
}

static void free_device_tables(dd_plan_s *p)
{
    if (p->d_span)
        cudaFree(p->d_span);
    if (p->d_rel)
        cudaFree(p->d_rel);
    if (p->d_zero)
        cudaFree(p->d_zero);
    if (p->d_prow)
        cudaFree(p->d_prow);
    if (p->d_gs_tab)
        cudaFree(p->d_gs_tab);
    p->d_span = p->d_rel = p->d_zero = p->d_prow = p->d_gs_tab = nullptr;
    p->uploaded = false;
}

// Uploads span/rel tables to the current device.  DD_ERR_CUDA when there is no usable device.
static dd_status upload_tables(dd_plan_s *p)
{
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess)
        return cuda_fail(e, "cudaGetDeviceCount");
    if (ndev <= 0)
        return cuda_fail(cudaErrorNoDevice, "cudaGetDeviceCount");
    free_device_tables(p);
    if ((e = cudaGetDevice(&p->device)) != cudaSuccess)
        return cuda_fail(e, "cudaGetDevice");
    const size_t span_bytes = p->span.size() * sizeof(SpanMeta), rel_bytes = p->rel.size();
    if ((e = cudaMalloc(&p->d_span, span_bytes)) != cudaSuccess)
        return cuda_fail(e, "cudaMalloc(span)");
    if ((e = cudaMalloc(&p->d_rel, rel_bytes)) != cudaSuccess) {
        free_device_tables(p);
        return cuda_fail(e, "cudaMalloc(rel)");
    }
    if (p->var.pad_chunks) {   // the all-zero span staged for padded channels
        if ((e = cudaMalloc(&p->d_zero, p->raw_slot)) != cudaSuccess ||
            (e = cudaMemset(p->d_zero, 0, p->raw_slot)) != cudaSuccess) {
            free_device_tables(p);
            return cuda_fail(e, "cudaMalloc(zero)");
        }
    }
    if ((e = cudaMemcpy(p->d_span, p->span.data(), span_bytes, cudaMemcpyHostToDevice)) != cudaSuccess ||
        (e = cudaMemcpy(p->d_rel, p->rel.data(), rel_bytes, cudaMemcpyHostToDevice)) != cudaSuccess) {
        free_device_tables(p);
        return cuda_fail(e, "cudaMemcpy(tables)");
    }
    if ((p->pairs || p->gr) && !p->prow.empty()) {   // variants 4 / 6: the channels and delay differences of every row
        const size_t pb = p->prow.size() * sizeof(int32_t);
        if ((e = cudaMalloc(&p->d_prow, pb)) != cudaSuccess ||
            (e = cudaMemcpy(p->d_prow, p->prow.data(), pb, cudaMemcpyHostToDevice)) != cudaSuccess) {
            free_device_tables(p);
            return cuda_fail(e, "cudaMalloc/Memcpy(pair rows)");
        }
    }
    if (p->gs && !p->gs_tab.empty()) {   // variant 5: the build entries of every stage
        const size_t tb = p->gs_tab.size() * sizeof(GsEntry);
        if ((e = cudaMalloc(&p->d_gs_tab, tb)) != cudaSuccess ||
            (e = cudaMemcpy(p->d_gs_tab, p->gs_tab.data(), tb, cudaMemcpyHostToDevice)) != cudaSuccess) {
            free_device_tables(p);
            return cuda_fail(e, "cudaMalloc/Memcpy(group-sum table)");
        }
    }
    p->uploaded = true;
    return DD_OK;
}

static void free_prof_events(dd_plan_s *p)
{
    for (void *e : p->prof_events)
        if (e)
            cudaEventDestroy(static_cast<cudaEvent_t>(e));
    p->prof_events.clear();
    p->prof_cap = p->prof_n = 0;
}

static int elem_size(int out_nbits)
{
    switch (out_nbits) {
    case DD_OUT_F32:
    case DD_OUT_U32:
        return 4;
    case DD_OUT_U16:
        return 2;
    case kOutU8:       // internal; check_execute rejects both at the C ABI
    case kOutPlanes:   // (sub-band intermediate: bit planes, one byte per sample)
        return 1;
    }
    return 0;
}

// Argument checks shared by dd_execute and dd_execute_host (pointer alignment is checked by the caller).
static dd_status check_execute(const dd_plan_s *p, int64_t nsamps, int64_t in_stride, int out_nbits)
{
    if (p->ndm <= 0)
        return DD_ERR_NO_DM_LIST;
    const int es = elem_size(out_nbits);
    if (nsamps <= 0 || es == 0 || out_nbits == kOutU8 || out_nbits == kOutPlanes)
        return DD_ERR_INVALID_ARG;
    if (in_stride <= 0 || in_stride % 16 != 0)
        return DD_ERR_ALIGNMENT;
    // in_stride*8 >= (nsamps + max_delay)*nbits, without overflow
    const int64_t need_bits_hi = (nsamps + p->max_delay);
    if (need_bits_hi > (INT64_MAX / 8) || in_stride > INT64_MAX / 8 || in_stride * 8 < need_bits_hi * p->nbits)
        return DD_ERR_STRIDE_TOO_SMALL;
    const int64_t vmax = (1 << p->nbits) - 1, top = static_cast<int64_t>(p->nlive) * vmax;   // over the summed channels
    if ((out_nbits == DD_OUT_U16 && top > 65535) || (out_nbits == DD_OUT_F32 && top >= (1 << 24)))
        return DD_ERR_OUT_RANGE;
    if (nsamps > (INT64_MAX / 8) / p->ndm)
        return DD_ERR_INVALID_ARG;
    return DD_OK;
}

// out_dm_stride: bytes between output rows, 0 = dense
static KernelParams make_params(const dd_plan_s *p, int64_t nsamps, const void *in, int64_t in_stride, void *out,
                                int out_nbits, int nbeams, int64_t in_beam_stride, int64_t out_beam_stride,
                                int64_t out_dm_stride = 0)
{
    KernelParams kp{};
    kp.in = static_cast<const uint8_t *>(in);
    kp.in_stride = in_stride;
    kp.in_row_bytes = in_stride;
    kp.in_beam_stride = in_beam_stride;
    kp.out = static_cast<uint8_t *>(out);
    kp.out_beam_stride = out_beam_stride;
    kp.nsamps = nsamps;
    kp.out_code = out_nbits;
    const int es = elem_size(out_nbits);
    const int vec_bytes = 4 * es;
    kp.out_dm_stride = out_dm_stride > 0 ? out_dm_stride : nsamps * es;
    auto aligned = [&](int64_t a) {   // every row starts on a multiple of a bytes
        return kp.out_dm_stride % a == 0 && reinterpret_cast<uintptr_t>(out) % a == 0 && out_beam_stride % a == 0;
    };
    kp.vec_ok = aligned(vec_bytes);
    kp.vec16_ok = aligned(16);
    kp.nchans = p->nlive;
    kp.nrows = p->nchans;
    kp.ndm = p->ndm;
    kp.nblk = p->nblk;
    kp.ntiles = static_cast<int32_t>((nsamps + p->var.TB - 1) / p->var.TB);
    kp.nbeams = nbeams;
    kp.cc = p->cc;
    kp.ngroups = p->ngroups;
    kp.group_cols = p->group_cols;
    kp.row_mul = 1;
    kp.in_blk_div = 0;
    kp.in_blk_stride = 0;
    // channels a CTA iterates over: the columns of one group (padded for the bit-plane kernel)
    kp.nchunks = ((p->var.pad_chunks ? p->group_cols : p->nlive) + p->cc - 1) / p->cc;
    kp.raw_slot = p->raw_slot;
    kp.lane_slot = p->lane_slot;
    kp.sub_slot = p->sub_slot;
    kp.nstages = p->nstages;
    kp.nchans_pad = p->nchans_pad;
    kp.zero = static_cast<const uint8_t *>(p->d_zero);
    kp.span = static_cast<const int4 *>(p->d_span);
    kp.rel = p->d_rel;
    return kp;
}

// Rebuilds delay table and tile metadata for (DM list, kill mask) into a scratch plan, then commits: a failure
// leaves the plan unchanged.  Uploads the tables when a device exists.
// The sub-band method on device-resident data ("two consecutive calls to the direct dedispersion
// routine and the addition of a temporary data buffer").  The temporary buffer is step 2's bit-plane work buffer:
// step 1 sums every sub-band for every nominal DM and stores the low 8 planes of its carry-save counters -- which
// ARE the 8-bit series S[beam][sub-band][nominal DM][t], t < nsamps + largest step-2 delay, in the layout step 2
// stages -- so that neither an output transpose, nor a byte buffer, nor a second pre-pass is needed; step 2
// dedisperses, for every group of trials, the miniature filterbank of its nominal DM.  Three kernels.
// dense_out: the output is a dense device slab [beam][d][nsamps] (the staging of dd_execute_host) instead of the
// caller's strides.
static dd_status execute_subband(dd_plan_s *plan, int64_t nsamps, const void *in_ptr, int64_t in_stride, void *out_ptr,
                                 int out_nbits, cudaStream_t st_, bool dense_out = false)
{
    dd_plan_s *s1 = plan->s1, *s2 = plan->s2;
    if (!s1 || !s2)
        return DD_ERR_INVALID_ARG;
    if (in_stride * 8 < (nsamps + plan->sb_extent) * plan->nbits)
        return DD_ERR_STRIDE_TOO_SMALL;
    dd_status st;
    for (dd_plan_s *q : {plan, s1, s2})
        if (!q->uploaded && (st = upload_tables(q)) != DD_OK)
            return st;
    const int nbeams = plan->nbeams, nsb = s2->nchans, ngrp = s1->ndm;
    const int64_t t1 = (nsamps + plan->sb_max_d2 + 31) / 32 * 32;
    cudaError_t e;
    // step 2's launch geometry first: N_SB channels; DM block blk reads the rows of nominal DM blk / (dm_group / 16)
    const int64_t out_beam = dense_out ? static_cast<int64_t>(plan->ndm) * nsamps * elem_size(out_nbits)
                                       : (nbeams > 1 ? plan->out_beam_stride : 0);
    KernelParams k2 = make_params(s2, nsamps, nullptr, 16, out_ptr, out_nbits, nbeams, 0, out_beam,
                                  dense_out ? 0 : plan->out_dm_stride);
    k2.nrows = nsb * ngrp;
    k2.row_mul = ngrp;
    k2.in_blk_div = plan->dm_group / s2->var.DB;
    BpWork w2;
    if ((e = bp_prepare_work(s2, k2, st_, true, &w2)) != cudaSuccess)
        return cuda_fail(e, "dd_execute sub-band work buffer");
    const bool prof = plan->prof_cap > 0 && plan->prof_n < plan->prof_cap;
    cudaEvent_t *ev = prof ? reinterpret_cast<cudaEvent_t *>(plan->prof_events.data()) + 3 * plan->prof_n : nullptr;
    if (prof)
        cudaEventRecord(ev[0], st_);
    // step 1: "DM trials" = the nominal DMs; a CTA sums gpc sub-bands one after the other (enough CTAs left to
    // fill the SMs a few times over), so that the copies of the next sub-band fly while this one is added
    const int64_t in_beam = nbeams > 1 ? plan->in_beam_stride : 0;
    KernelParams k1 = make_params(s1, t1, in_ptr, in_stride, s2->d_work, kOutPlanes, nbeams, in_beam, 0);
    k1.pl_conv = w2.conv;
    k1.pl_beam = w2.w_beam;
    k1.pl_units = static_cast<int32_t>(w2.units);
    int sms = 148;
    (void)cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, plan->device >= 0 ? plan->device : 0);
    const int64_t ctas1 = static_cast<int64_t>(k1.nblk) * k1.ntiles * nbeams * k1.ngroups;
    int64_t gpc = ctas1 / (8 * static_cast<int64_t>(sms));   // measured on the cfg2 shape: flat from 4 to 16 sub-bands per CTA
    if (plan->sb_gpc > 0)   // dd_set_tuning(DD_TUNE_SUBBAND_GPC)
        gpc = plan->sb_gpc;
    k1.gpc = static_cast<int32_t>(std::max<int64_t>(1, std::min<int64_t>(gpc, k1.ngroups)));
    s1->prof_mid = nullptr;
    if ((e = launch_direct(s1, k1, st_)) != cudaSuccess)
        return cuda_fail(e, "dd_execute sub-band step 1");
    s2->prof_mid = prof ? ev[1] : nullptr;
    e = launch_variant3(s2, k2, st_, true);
    s2->prof_mid = nullptr;
    if (e != cudaSuccess)
        return cuda_fail(e, "dd_execute sub-band step 2");
    if (prof) {
        cudaEventRecord(ev[2], st_);
        ++plan->prof_n;
    }
    plan->last_launches = launches_per_execute(s1) + 1;
    return DD_OK;
}

static void destroy_subplan(dd_plan_s *q)
{
    if (!q)
        return;
    free_device_tables(q);
    if (q->d_work)
        cudaFree(q->d_work);
    delete q;
}

static dd_status replan(dd_plan_s *plan, std::vector<double> dm, std::vector<uint8_t> keep, int sb_nchans, int dm_group)
{
    dd_plan_s scratch;
    scratch.sb_nchans = sb_nchans;
    scratch.dm_group = dm_group;
    scratch.nchans = plan->nchans;
    scratch.dt = plan->dt;
    scratch.f_top = plan->f_top;
    scratch.df = plan->df;
    scratch.nbits = plan->nbits;
    scratch.ndm = static_cast<int>(dm.size());
    scratch.force_variant = plan->force_variant;
    scratch.in_planes = plan->in_planes;   // dd_set_input_max: keeps the plan on the plane-skipping kernel
    scratch.gs_force_G = plan->gs_force_G;
    scratch.gs_force_cc = plan->gs_force_cc;
    scratch.dm.swap(dm);
    scratch.keep.swap(keep);
    dd_status st = compute_delay_table(&scratch);
    if (st != DD_OK)
        return st;
    st = build_tiles(&scratch);
    if (st != DD_OK)
        return st;
    dd_plan_s *s1 = nullptr, *s2 = nullptr;
    if (sb_nchans > 0) {   // the two direct steps of the sub-band method
        s1 = new dd_plan_s();
        s2 = new dd_plan_s();
        st = build_subband(&scratch, s1, s2, &scratch.sb_nominal, &scratch.sb_max_d2, &scratch.sb_extent);
        if (st == DD_OK && (!s1->var.bitplane || !s2->var.bitplane))
            st = DD_ERR_SMEM;
        if (st != DD_OK) {
            delete s1;
            delete s2;
            return st;
        }
    }
    free_device_tables(plan);
    destroy_subplan(plan->s1);
    destroy_subplan(plan->s2);
    plan->s1 = s1;
    plan->s2 = s2;
    for (dd_plan_s *q : {s1, s2})
        if (q)
            q->bp_tpc = plan->bp_tpc;
    plan->sb_nchans = sb_nchans;
    plan->dm_group = dm_group;
    plan->sb_nominal.swap(scratch.sb_nominal);
    plan->sb_max_d2 = scratch.sb_max_d2;
    plan->sb_extent = sb_nchans > 0 ? scratch.sb_extent : -1;
    plan->ndm = scratch.ndm;
    plan->dm.swap(scratch.dm);
    plan->keep.swap(scratch.keep);
    plan->live.swap(scratch.live);
    plan->nlive = scratch.nlive;
    plan->delay.swap(scratch.delay);
    plan->max_delay = scratch.max_delay;
    plan->var = scratch.var;
    plan->nblk = scratch.nblk;
    plan->cc = scratch.cc;
    plan->nchans_pad = scratch.nchans_pad;
    plan->ngroups = scratch.ngroups;
    plan->group_cols = scratch.group_cols;
    plan->nstages = scratch.nstages;
    plan->patch = scratch.patch;
    plan->long_mode = scratch.long_mode;
    plan->max_span_end = scratch.max_span_end;
    plan->raw_slot = scratch.raw_slot;
    plan->sub_slot = scratch.sub_slot;
    plan->lane_slot = scratch.lane_slot;
    plan->smem_bytes = scratch.smem_bytes;
    plan->final32 = scratch.final32;
    plan->span.swap(scratch.span);
    plan->rel.swap(scratch.rel);
    plan->pairs = scratch.pairs;
    plan->pair_nbits = scratch.pair_nbits;
    plan->pair_planes = scratch.pair_planes;
    plan->rows_per_chunk = scratch.rows_per_chunk;
    plan->prow.swap(scratch.prow);
    plan->n_prows = scratch.n_prows;
    plan->gr = scratch.gr;
    plan->gr_stage_slots = scratch.gr_stage_slots;
    plan->gs = scratch.gs;
    plan->gs_G = scratch.gs_G;
    plan->gs_rows = scratch.gs_rows;
    plan->gs_row_units = scratch.gs_row_units;
    plan->gs_raw_sub = scratch.gs_raw_sub;
    plan->gs_nsr = scratch.gs_nsr;
    plan->gs_nsp = scratch.gs_nsp;
    plan->gs_patch = scratch.gs_patch;
    plan->gs_tab.swap(scratch.gs_tab);
    plan->pair_geom[2] = 0;
    plan->last_launches = 0;
    // upload now when a device exists; otherwise the first dd_execute retries (documented in dd.h)
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) == cudaSuccess && ndev > 0) {
        st = upload_tables(plan);
        if (st == DD_OK && plan->s1)
            st = upload_tables(plan->s1);
        if (st == DD_OK && plan->s2)
            st = upload_tables(plan->s2);
        if (st != DD_OK)
            return st;
    } else {
        (void)cudaGetLastError();
    }
    return DD_OK;
}

}  // namespace dd

using namespace dd;

extern "C" {

dd_status dd_plan_create(dd_plan *plan, int nchans, double dt, double f_top, double df, int nbits)
{
    if (!plan)
        return DD_ERR_NULL;
    *plan = nullptr;
    if (nchans <= 0 || !(dt > 0.0) || !std::isfinite(dt) || !(f_top > 0.0) || !std::isfinite(f_top) || !(df < 0.0) ||
        !std::isfinite(df) || (nbits != 2 && nbits != 4 && nbits != 8))
        return DD_ERR_INVALID_ARG;
    if (!(f_top + static_cast<double>(nchans - 1) * df > 0.0))
        return DD_ERR_INVALID_ARG;
    dd_plan_s *p = new (std::nothrow) dd_plan_s();
    if (!p)
        return DD_ERR_NOMEM;
    p->nchans = nchans;
    p->dt = dt;
    p->f_top = f_top;
    p->df = df;
    p->nbits = nbits;
    *plan = p;
    return DD_OK;
}

dd_status dd_plan_destroy(dd_plan plan)
{
    if (!plan)
        return DD_OK;
    free_device_tables(plan);
    if (plan->d_work)
        cudaFree(plan->d_work);
    if (plan->d_pairwork)
        cudaFree(plan->d_pairwork);
    for (void *st : plan->pair_streams)
        if (st)
            cudaStreamDestroy(static_cast<cudaStream_t>(st));
    for (void *ev : plan->pair_events)
        if (ev)
            cudaEventDestroy(static_cast<cudaEvent_t>(ev));
    if (plan->d_tmp)
        cudaFree(plan->d_tmp);
    destroy_subplan(plan->s1);
    destroy_subplan(plan->s2);
    free_stage(plan->stage);
    free_prof_events(plan);
    delete plan;
    return DD_OK;
}

dd_status dd_set_dm_list(dd_plan plan, const double *dm_list, int ndm)
{
    if (!plan || !dm_list)
        return DD_ERR_NULL;
    if (ndm <= 0)
        return DD_ERR_INVALID_ARG;
    for (int d = 0; d < ndm; ++d)
        if (!std::isfinite(dm_list[d]) || dm_list[d] < 0.0)
            return DD_ERR_INVALID_ARG;
    try {
        return replan(plan, std::vector<double>(dm_list, dm_list + ndm), plan->keep, plan->sb_nchans, plan->dm_group);
    } catch (const std::bad_alloc &) {
        return DD_ERR_NOMEM;
    }
}

dd_status dd_set_killmask(dd_plan plan, const int32_t *mask)
{
    if (!plan)
        return DD_ERR_NULL;
    try {
        std::vector<uint8_t> keep;
        if (mask) {
            keep.resize(plan->nchans);
            for (int c = 0; c < plan->nchans; ++c)
                keep[c] = mask[c] != 0;
        }
        if (plan->ndm <= 0) {   // no DM list yet: remembered, applied by dd_set_dm_list
            plan->keep.swap(keep);
            return DD_OK;
        }
        return replan(plan, plan->dm, keep, plan->sb_nchans, plan->dm_group);
    } catch (const std::bad_alloc &) {
        return DD_ERR_NOMEM;
    }
}

dd_status dd_set_subband(dd_plan plan, int sb_nchans, int dm_group)
{
    if (!plan)
        return DD_ERR_NULL;
    if (sb_nchans == 0 && dm_group == 0) {   // back to the direct transform
        if (plan->ndm <= 0) {
            plan->sb_nchans = plan->dm_group = 0;
            return DD_OK;
        }
    } else {
        if (sb_nchans < 1 || dm_group < 1 || plan->nchans % sb_nchans != 0 || dm_group % 16 != 0)
            return DD_ERR_INVALID_ARG;
        if (static_cast<int64_t>(sb_nchans) * ((1 << plan->nbits) - 1) > 255)
            return DD_ERR_OUT_RANGE;   // the intermediate series are kept in 8 bits
        if (plan->ndm <= 0) {
            plan->sb_nchans = sb_nchans;
            plan->dm_group = dm_group;
            return DD_OK;
        }
    }
    try {
        return replan(plan, plan->dm, plan->keep, sb_nchans, dm_group);
    } catch (const std::bad_alloc &) {
        return DD_ERR_NOMEM;
    }
}

int64_t dd_get_subband_extent(dd_plan plan)
{
    if (!plan)
        return DD_ERR_NULL;
    if (plan->ndm <= 0)
        return DD_ERR_NO_DM_LIST;
    if (plan->sb_nchans <= 0)
        return DD_ERR_INVALID_ARG;
    return plan->sb_extent;
}

dd_status dd_get_subband_tables(dd_plan plan, int32_t *nominal, int32_t *delta1, int32_t *delta2)
{
    if (!plan)
        return DD_ERR_NULL;
    if (plan->ndm <= 0)
        return DD_ERR_NO_DM_LIST;
    if (plan->sb_nchans <= 0 || !plan->s1 || !plan->s2)
        return DD_ERR_INVALID_ARG;
    if (nominal)
        std::memcpy(nominal, plan->sb_nominal.data(), plan->sb_nominal.size() * sizeof(int32_t));
    if (delta1)
        std::memcpy(delta1, plan->s1->delay.data(), plan->s1->delay.size() * sizeof(int32_t));
    if (delta2)
        std::memcpy(delta2, plan->s2->delay.data(), plan->s2->delay.size() * sizeof(int32_t));
    return DD_OK;
}

dd_status dd_get_delay_table(dd_plan plan, int32_t *table)
{
    if (!plan || !table)
        return DD_ERR_NULL;
    if (plan->ndm <= 0)
        return DD_ERR_NO_DM_LIST;
    std::memcpy(table, plan->delay.data(), plan->delay.size() * sizeof(int32_t));
    return DD_OK;
}

int64_t dd_get_max_delay(dd_plan plan)
{
    if (!plan)
        return DD_ERR_NULL;
    if (plan->ndm <= 0)
        return DD_ERR_NO_DM_LIST;
    return plan->max_delay;
}

dd_status dd_set_batch(dd_plan plan, int nbeams, int64_t in_beam_stride, int64_t out_beam_stride)
{
    if (!plan)
        return DD_ERR_NULL;
    if (nbeams <= 0 || in_beam_stride < 0 || out_beam_stride < 0)
        return DD_ERR_INVALID_ARG;
    if (nbeams > 1 && in_beam_stride % 16 != 0)
        return DD_ERR_ALIGNMENT;
    plan->nbeams = nbeams;
    plan->in_beam_stride = nbeams > 1 ? in_beam_stride : 0;
    plan->out_beam_stride = nbeams > 1 ? out_beam_stride : 0;
    return DD_OK;
}

dd_status dd_execute(dd_plan plan, int64_t nsamps, const void *in_ptr, int64_t in_stride, void *out_ptr, int out_nbits,
                     void *stream)
{
    if (!plan || !in_ptr || !out_ptr)
        return DD_ERR_NULL;
    dd_status st = check_execute(plan, nsamps, in_stride, out_nbits);
    if (st != DD_OK)
        return st;
    const int es = elem_size(out_nbits);
    if (reinterpret_cast<uintptr_t>(in_ptr) % 16 != 0 || reinterpret_cast<uintptr_t>(out_ptr) % es != 0)
        return DD_ERR_ALIGNMENT;
    const int64_t pitch = plan->out_dm_stride > 0 ? plan->out_dm_stride : nsamps * es;   // bytes between output rows
    if (pitch % es != 0)
        return DD_ERR_ALIGNMENT;
    if (pitch < nsamps * es)
        return DD_ERR_STRIDE_TOO_SMALL;
    if (plan->nbeams > 1) {
        if (plan->out_beam_stride % es != 0)
            return DD_ERR_ALIGNMENT;
        if (plan->in_beam_stride < static_cast<int64_t>(plan->nchans) * in_stride ||
            plan->out_beam_stride < static_cast<int64_t>(plan->ndm - 1) * pitch + nsamps * es)
            return DD_ERR_STRIDE_TOO_SMALL;
    }
    cudaStream_t st_ = static_cast<cudaStream_t>(stream);
    if (plan->nlive == 0) {   // every channel killed: the sums are zero (float32 zero is all-zero bits too)
        for (int b = 0; b < plan->nbeams; ++b) {
            uint8_t *o = static_cast<uint8_t *>(out_ptr) + static_cast<int64_t>(b) * (plan->nbeams > 1 ? plan->out_beam_stride : 0);
            const cudaError_t me = cudaMemset2DAsync(o, static_cast<size_t>(pitch), 0, static_cast<size_t>(nsamps) * es,
                                                     static_cast<size_t>(plan->ndm), st_);
            if (me != cudaSuccess)
                return cuda_fail(me, "dd_execute memset");
        }
        plan->last_launches = 0;
        return DD_OK;
    }
    if (plan->sb_nchans > 0)
        return execute_subband(plan, nsamps, in_ptr, in_stride, out_ptr, out_nbits, st_);
    if (!plan->uploaded) {
        st = upload_tables(plan);
        if (st != DD_OK)
            return st;
    }
    const KernelParams kp = make_params(plan, nsamps, in_ptr, in_stride, out_ptr, out_nbits, plan->nbeams,
                                        plan->in_beam_stride, plan->out_beam_stride, plan->out_dm_stride);
    const bool prof = plan->prof_cap > 0 && plan->prof_n < plan->prof_cap;
    cudaEvent_t *ev = prof ? reinterpret_cast<cudaEvent_t *>(plan->prof_events.data()) + 3 * plan->prof_n : nullptr;
    plan->prof_mid = nullptr;
    if (prof) {
        cudaEventRecord(ev[0], st_);
        if (plan->var.bitplane)
            plan->prof_mid = ev[1];        // recorded by the launcher after the pre-pass
        else
            cudaEventRecord(ev[1], st_);
    }
    const cudaError_t e = launch_direct(plan, kp, st_);
    plan->prof_mid = nullptr;
    if (e != cudaSuccess)
        return cuda_fail(e, "dd_execute launch");
    if (prof) {
        cudaEventRecord(ev[2], st_);
        ++plan->prof_n;
    }
    plan->last_launches = launches_per_execute(plan);
    return DD_OK;
}

// dd_execute without allocations (include/dd.h): the argument checks of dd_execute, then the bit-plane kernel on the
// library's fixed scratch array.  Nothing here, or below it, calls cudaMalloc / cudaFree.
dd_status dd_execute_static(dd_plan plan, int64_t nsamps, const void *in_ptr, int64_t in_stride, void *out_ptr,
                            int out_nbits, void *stream)
{
    if (!plan || !in_ptr || !out_ptr)
        return DD_ERR_NULL;
    dd_status st = check_execute(plan, nsamps, in_stride, out_nbits);
    if (st != DD_OK)
        return st;
    const int es = elem_size(out_nbits);
    if (reinterpret_cast<uintptr_t>(in_ptr) % 16 != 0 || reinterpret_cast<uintptr_t>(out_ptr) % es != 0)
        return DD_ERR_ALIGNMENT;
    const int64_t pitch = plan->out_dm_stride > 0 ? plan->out_dm_stride : nsamps * es;
    if (pitch % es != 0)
        return DD_ERR_ALIGNMENT;
    if (pitch < nsamps * es)
        return DD_ERR_STRIDE_TOO_SMALL;
    if (plan->nbeams > 1) {
        if (plan->out_beam_stride % es != 0)
            return DD_ERR_ALIGNMENT;
        if (plan->in_beam_stride < static_cast<int64_t>(plan->nchans) * in_stride ||
            plan->out_beam_stride < static_cast<int64_t>(plan->ndm - 1) * pitch + nsamps * es)
            return DD_ERR_STRIDE_TOO_SMALL;
    }
    cudaStream_t st_ = static_cast<cudaStream_t>(stream);
    if (plan->nlive == 0) {   // every channel killed: zeros, no scratch
        for (int b = 0; b < plan->nbeams; ++b) {
            uint8_t *o = static_cast<uint8_t *>(out_ptr) + static_cast<int64_t>(b) * (plan->nbeams > 1 ? plan->out_beam_stride : 0);
            const cudaError_t me = cudaMemset2DAsync(o, static_cast<size_t>(pitch), 0, static_cast<size_t>(nsamps) * es,
                                                     static_cast<size_t>(plan->ndm), st_);
            if (me != cudaSuccess)
                return cuda_fail(me, "dd_execute_static memset");
        }
        plan->last_launches = 0;
        return DD_OK;
    }
    if (plan->sb_nchans > 0 || plan->var.id != 3 || !plan->var.bitplane) {
        g_cuda_error = "dd_execute_static: the plan must run kernel variant 3 (dd_set_kernel_variant(plan, 3) before dd_set_dm_list) "
                       "without the sub-band method";
        return DD_ERR_UNSUPPORTED;
    }
    int dev = -1;
    const cudaError_t de = cudaGetDevice(&dev);
    if (de != cudaSuccess)
        return cuda_fail(de, "dd_execute_static cudaGetDevice");
    if (!plan->uploaded || plan->device != dev) {   // (uploading would allocate)
        g_cuda_error = "dd_execute_static: the plan's tables are not on the current device (call dd_set_dm_list with this device current)";
        return DD_ERR_UNSUPPORTED;
    }
    const KernelParams kp = make_params(plan, nsamps, in_ptr, in_stride, out_ptr, out_nbits, plan->nbeams,
                                        plan->in_beam_stride, plan->out_beam_stride, plan->out_dm_stride);
    const size_t need = static_work_need(plan, kp);
    if (need > static_cast<size_t>(DD_STATIC_WORKSPACE_BYTES)) {
        g_cuda_error = "dd_execute_static: the call needs " + std::to_string(need) + " bytes of scratch, the static array holds " +
                       std::to_string(static_cast<size_t>(DD_STATIC_WORKSPACE_BYTES)) + " (DD_STATIC_WORKSPACE_BYTES)";
        return DD_ERR_TOO_LARGE;
    }
    plan->prof_mid = nullptr;
    const cudaError_t e = launch_variant3_static(plan, kp, st_);
    if (e != cudaSuccess)
        return cuda_fail(e, "dd_execute_static launch");
    plan->last_launches = 2;
    return DD_OK;
}

dd_status dd_execute_host(dd_plan plan, int64_t nsamps, const void *in_host, int64_t in_stride, void *out_host,
                          int out_nbits)
{
    if (!plan || !in_host || !out_host)
        return DD_ERR_NULL;
    dd_status st = check_execute(plan, nsamps, in_stride, out_nbits);
    if (st != DD_OK)
        return st;
    const int es = elem_size(out_nbits);
    if (plan->sb_nchans > 0 && in_stride * 8 < (nsamps + plan->sb_extent) * plan->nbits)
        return DD_ERR_STRIDE_TOO_SMALL;   // the two steps read sb_extent samples beyond nsamps
    const int64_t row_pitch = plan->out_dm_stride > 0 ? plan->out_dm_stride : nsamps * es;   // host rows (dd_set_output_stride)
    if (row_pitch % es != 0)
        return DD_ERR_ALIGNMENT;
    if (row_pitch < nsamps * es)
        return DD_ERR_STRIDE_TOO_SMALL;
    const int64_t beam_span = static_cast<int64_t>(plan->ndm - 1) * row_pitch + nsamps * es;   // bytes a beam's rows cover
    if (plan->nlive == 0) {   // every channel killed
        const int64_t pitch = plan->nbeams > 1 ? plan->out_beam_stride : 0;
        if (plan->nbeams > 1 && pitch < beam_span)
            return DD_ERR_STRIDE_TOO_SMALL;
        for (int b = 0; b < plan->nbeams; ++b)
            for (int d = 0; d < plan->ndm; ++d)
                std::memset(static_cast<uint8_t *>(out_host) + b * pitch + d * row_pitch, 0, static_cast<size_t>(nsamps) * es);
        plan->last_launches = 0;
        return DD_OK;
    }
    if (!plan->uploaded) {
        st = upload_tables(plan);
        if (st != DD_OK)
            return st;
    }
    const int nbeams = plan->nbeams;
    const int64_t in_beam = nbeams > 1 ? plan->in_beam_stride : static_cast<int64_t>(plan->nchans) * in_stride;
    const int64_t out_beam_host = nbeams > 1 ? plan->out_beam_stride : static_cast<int64_t>(plan->ndm) * row_pitch;
    if (nbeams > 1 && (in_beam < static_cast<int64_t>(plan->nchans) * in_stride || out_beam_host < beam_span))
        return DD_ERR_STRIDE_TOO_SMALL;

    // Time slabs: the input slab of output samples [s0, s0+len) is rows [s0, s0+len+max_delay); the slab
    // length is a multiple of the tile so that slab starts stay 16-byte aligned in the packed rows.
    const int64_t TB = plan->var.TB;
    int64_t slab = ((plan->host_slab > 0 ? static_cast<int64_t>(plan->host_slab) : (int64_t(1) << 15)) + TB - 1) / TB * TB;
    if (slab > (nsamps + TB - 1) / TB * TB || plan->sb_nchans > 0)   // the sub-band method runs as one slab (its
        slab = (nsamps + TB - 1) / TB * TB;                          // intermediate series span the whole call)
    const int64_t nslabs = (nsamps + slab - 1) / slab;
    const size_t in_bytes = static_cast<size_t>(in_beam) * nbeams;
    const size_t out_slab_bytes = static_cast<size_t>(nbeams) * plan->ndm * slab * es;

    cudaError_t e;
    if (!plan->stage)
        plan->stage = new (std::nothrow) HostStage();
    HostStage *S = plan->stage;
    if (!S)
        return DD_ERR_NOMEM;
    if (!S->streams) {
        if ((e = cudaStreamCreateWithFlags(&S->copy_in, cudaStreamNonBlocking)) != cudaSuccess ||
            (e = cudaStreamCreateWithFlags(&S->compute, cudaStreamNonBlocking)) != cudaSuccess ||
            (e = cudaStreamCreateWithFlags(&S->copy_out[0], cudaStreamNonBlocking)) != cudaSuccess ||
            (e = cudaStreamCreateWithFlags(&S->copy_out[1], cudaStreamNonBlocking)) != cudaSuccess)
            return cuda_fail(e, "cudaStreamCreate");
        cudaEventCreateWithFlags(&S->in_ready, cudaEventDisableTiming);
        cudaEventCreateWithFlags(&S->in_rest, cudaEventDisableTiming);
        for (int i = 0; i < 2; ++i) {
            cudaEventCreateWithFlags(&S->done[i], cudaEventDisableTiming);
            cudaEventCreateWithFlags(&S->drained[i], cudaEventDisableTiming);
        }
        S->streams = true;
    }
    if (S->in_bytes < in_bytes) {
        cudaFree(S->d_in);
        S->d_in = nullptr;
        S->in_bytes = 0;
        if ((e = cudaMalloc(&S->d_in, in_bytes)) != cudaSuccess)
            return cuda_fail(e, "cudaMalloc(stage in)");
        S->in_bytes = in_bytes;
    }
    if (S->out_bytes < out_slab_bytes) {
        for (int i = 0; i < 2; ++i) {
            cudaFree(S->d_out[i]);
            S->d_out[i] = nullptr;
        }
        S->out_bytes = 0;
        for (int i = 0; i < 2; ++i)
            if ((e = cudaMalloc(&S->d_out[i], out_slab_bytes)) != cudaSuccess)
                return cuda_fail(e, "cudaMalloc(stage out)");
        S->out_bytes = out_slab_bytes;
    }

    // input (5-30x smaller than the output): first the bytes of every row that the first slab reads, so that its kernels --
    // and, behind them, the first copy out, which is what the call is bound by -- start early; then the rest of the rows
    const int64_t nrows_all = static_cast<int64_t>(nbeams) * plan->nchans;
    const bool rows_dense = nbeams == 1 || in_beam == static_cast<int64_t>(plan->nchans) * in_stride;
    // (the kernels of a slab of n tiles read n - 1 tiles + max_span_end samples of every row, in whole 16-byte groups)
    const int64_t reach = std::max<int64_t>(plan->max_span_end, TB + plan->max_delay);
    int64_t head = ((slab - TB + reach + 256) * plan->nbits / 8 + 15) / 16 * 16;
    if (!rows_dense || nslabs < 2 || head >= in_stride)
        head = 0;   // (one copy of everything)
    if (head > 0) {
        if ((e = cudaMemcpy2DAsync(S->d_in, static_cast<size_t>(in_stride), in_host, static_cast<size_t>(in_stride),
                                   static_cast<size_t>(head), static_cast<size_t>(nrows_all), cudaMemcpyHostToDevice,
                                   S->copy_in)) != cudaSuccess)
            return cuda_fail(e, "cudaMemcpy2DAsync(in, head)");
        cudaEventRecord(S->in_ready, S->copy_in);
        if ((e = cudaMemcpy2DAsync(S->d_in + head, static_cast<size_t>(in_stride), static_cast<const uint8_t *>(in_host) + head,
                                   static_cast<size_t>(in_stride), static_cast<size_t>(in_stride - head),
                                   static_cast<size_t>(nrows_all), cudaMemcpyHostToDevice, S->copy_in)) != cudaSuccess) {
            cudaStreamSynchronize(S->copy_in);
            return cuda_fail(e, "cudaMemcpy2DAsync(in, rest)");
        }
        cudaEventRecord(S->in_rest, S->copy_in);
    } else {
        if ((e = cudaMemcpyAsync(S->d_in, in_host, in_bytes, cudaMemcpyHostToDevice, S->copy_in)) != cudaSuccess)
            return cuda_fail(e, "cudaMemcpyAsync(in)");
        cudaEventRecord(S->in_ready, S->copy_in);
        cudaEventRecord(S->in_rest, S->copy_in);
    }
    cudaStreamWaitEvent(S->compute, S->in_ready, 0);

    // an error below must not return while copies into the caller's buffers are still in flight
    auto fail_drained = [&](dd_status code) {
        cudaStreamSynchronize(S->copy_in);
        cudaStreamSynchronize(S->compute);
        cudaStreamSynchronize(S->copy_out[0]);
        cudaStreamSynchronize(S->copy_out[1]);
        (void)cudaGetLastError();
        return code;
    };
    int64_t launches = 0;
    for (int64_t k = 0; k < nslabs; ++k) {
        const int b = static_cast<int>(k & 1);
        const int64_t s0 = k * slab, len = (s0 + slab <= nsamps) ? slab : nsamps - s0;
        if (k == 1)
            cudaStreamWaitEvent(S->compute, S->in_rest, 0);      // the rest of the input rows
        if (k >= 2)
            cudaStreamWaitEvent(S->compute, S->drained[b], 0);   // slab buffer b has been copied out
        const uint8_t *in_slab = S->d_in + (s0 * plan->nbits) / 8;
        if (plan->sb_nchans > 0) {   // PAPER.md:317-321 on the staged copy (one slab)
            const int64_t keep_beam = plan->in_beam_stride;
            plan->in_beam_stride = in_beam;
            const dd_status sst = execute_subband(plan, len, in_slab, in_stride, S->d_out[b], out_nbits, S->compute, true);
            plan->in_beam_stride = keep_beam;
            if (sst != DD_OK)
                return fail_drained(sst);
            launches += plan->last_launches;
        } else {
            KernelParams kp = make_params(plan, len, in_slab, in_stride, S->d_out[b], out_nbits, nbeams, in_beam,
                                          static_cast<int64_t>(plan->ndm) * len * es);
            kp.in_row_bytes = in_stride - (s0 * plan->nbits) / 8;
            if ((e = launch_direct(plan, kp, S->compute)) != cudaSuccess)
                return fail_drained(cuda_fail(e, "dd_execute_host launch"));
            launches += launches_per_execute(plan);
        }
        cudaEventRecord(S->done[b], S->compute);
        cudaStreamWaitEvent(S->copy_out[b], S->done[b], 0);
        for (int beam = 0; beam < nbeams; ++beam) {
            uint8_t *dst = static_cast<uint8_t *>(out_host) + static_cast<size_t>(beam) * out_beam_host + s0 * es;
            const uint8_t *src = S->d_out[b] + static_cast<size_t>(beam) * plan->ndm * len * es;
            if ((e = cudaMemcpy2DAsync(dst, static_cast<size_t>(row_pitch), src, static_cast<size_t>(len) * es,
                                       static_cast<size_t>(len) * es, plan->ndm, cudaMemcpyDeviceToHost,
                                       S->copy_out[b])) != cudaSuccess)
                return fail_drained(cuda_fail(e, "cudaMemcpy2DAsync(out)"));
        }
        cudaEventRecord(S->drained[b], S->copy_out[b]);
    }
    for (int i = 0; i < 2; ++i)
        if ((e = cudaStreamSynchronize(S->copy_out[i])) != cudaSuccess)
            return cuda_fail(e, "cudaStreamSynchronize(out)");
    if ((e = cudaStreamSynchronize(S->compute)) != cudaSuccess)
        return cuda_fail(e, "cudaStreamSynchronize(compute)");
    plan->last_launches = launches;
    return DD_OK;
}

dd_status dd_time_scrunch(int nrows, int64_t nsamps_out, const void *in_ptr, int64_t in_stride, int nbits_in, void *out_ptr,
                          int64_t out_stride, int nbits_out, void *stream)
{
    if (!in_ptr || !out_ptr)
        return DD_ERR_NULL;
    if (nrows <= 0 || nsamps_out <= 0 || (nbits_in != 2 && nbits_in != 4 && nbits_in != 8) ||
        (nbits_out != 2 && nbits_out != 4 && nbits_out != 8))
        return DD_ERR_INVALID_ARG;
    if (2 * ((1 << nbits_in) - 1) > (1 << nbits_out) - 1)
        return DD_ERR_OUT_RANGE;   // the pair sums do not fit the output width (8-bit input has no wider packed width)
    if (reinterpret_cast<uintptr_t>(in_ptr) % 16 != 0 || reinterpret_cast<uintptr_t>(out_ptr) % 16 != 0 || in_stride % 16 != 0 ||
        out_stride % 16 != 0)
        return DD_ERR_ALIGNMENT;
    if (nsamps_out > (INT64_MAX / 64))
        return DD_ERR_INVALID_ARG;
    const int64_t out_bytes = ((nsamps_out * nbits_out + 7) / 8 + 15) / 16 * 16;
    const int64_t in_bytes = out_bytes * 2 * nbits_in / nbits_out;   // whole 16-byte groups of the input are read
    if (out_stride < out_bytes || in_stride < in_bytes)
        return DD_ERR_STRIDE_TOO_SMALL;
    const cudaError_t e = launch_scrunch(nbits_in, nbits_out, nrows, static_cast<const uint8_t *>(in_ptr), in_stride,
                                         static_cast<uint8_t *>(out_ptr), out_stride, out_bytes, static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess)
        return cuda_fail(e, "dd_time_scrunch launch");
    return DD_OK;
}

dd_status dd_set_output_stride(dd_plan plan, int64_t out_dm_stride)
{
    if (!plan)
        return DD_ERR_NULL;
    if (out_dm_stride < 0)
        return DD_ERR_INVALID_ARG;
    plan->out_dm_stride = out_dm_stride;
    return DD_OK;
}

dd_status dd_set_input_max(dd_plan plan, int vmax)
{
    if (!plan)
        return DD_ERR_NULL;
    if (vmax < 0 || vmax > (1 << plan->nbits) - 1)
        return DD_ERR_INVALID_ARG;
    int planes = 0;
    while (vmax >> planes)
        ++planes;
    if (planes == plan->in_planes)
        return DD_OK;
    const int before = plan->in_planes;
    plan->in_planes = planes;   // 0 = all nbits planes
    if (plan->ndm <= 0)
        return DD_OK;
    // the promise decides which kernel serves the plan (variant 3 skips planes, variant 4 does not): plan again
    try {
        const dd_status st = replan(plan, plan->dm, plan->keep, plan->sb_nchans, plan->dm_group);
        if (st != DD_OK)
            plan->in_planes = before;
        return st;
    } catch (const std::bad_alloc &) {
        plan->in_planes = before;
        return DD_ERR_NOMEM;
    }
}

dd_status dd_set_kernel_variant(dd_plan plan, int variant)
{
    if (!plan)
        return DD_ERR_NULL;
    if (variant < 0 || variant > 6)
        return DD_ERR_INVALID_ARG;
    plan->force_variant = variant;
    return DD_OK;
}

dd_status dd_set_tuning(dd_plan plan, int key, int value)
{
    if (!plan)
        return DD_ERR_NULL;
    if (value < 0)
        return DD_ERR_INVALID_ARG;
    switch (key) {
    case DD_TUNE_SUBBAND_GPC:
        plan->sb_gpc = value;
        return DD_OK;
    case DD_TUNE_GROUP_SIZE:
        if (value != 0 && value != 2 && value != 4)
            return DD_ERR_INVALID_ARG;
        plan->gs_force_G = value;
        return DD_OK;
    case DD_TUNE_GROUPS_PER_STAGE:
        plan->gs_force_cc = value;
        return DD_OK;
    case DD_TUNE_PAIR_TILES:
        plan->pair_tiles = value;
        return DD_OK;
    case DD_TUNE_HOST_SLAB:
        plan->host_slab = value;
        return DD_OK;
    case DD_TUNE_TILES_PER_CTA:
        plan->bp_tpc = value;
        for (dd_plan_s *q : {plan->s1, plan->s2})
            if (q)
                q->bp_tpc = value;
        return DD_OK;
    }
    return DD_ERR_INVALID_ARG;
}

dd_status dd_set_workspace_limit(dd_plan plan, int64_t bytes)
{
    if (!plan)
        return DD_ERR_NULL;
    if (bytes < 0)
        return DD_ERR_INVALID_ARG;
    plan->ws_limit = bytes;
    plan->pair_geom[2] = 0;   // worked out again at the next dd_execute
    return DD_OK;
}

int64_t dd_get_workspace_bytes(dd_plan plan)
{
    if (!plan)
        return DD_ERR_NULL;
    int64_t b = static_cast<int64_t>(plan->work_bytes) + static_cast<int64_t>(plan->pairwork_bytes);
    for (const dd_plan_s *q : {plan->s1, plan->s2})
        if (q)
            b += static_cast<int64_t>(q->work_bytes);
    if (plan->stage)
        b += static_cast<int64_t>(plan->stage->in_bytes) + 2 * static_cast<int64_t>(plan->stage->out_bytes);
    return b;
}

dd_status dd_get_launch_info(dd_plan plan, int64_t *info)
{
    if (!plan || !info)
        return DD_ERR_NULL;
    if (plan->ndm <= 0)
        return DD_ERR_NO_DM_LIST;
    info[0] = plan->var.DB;
    info[1] = plan->var.TB;
    info[2] = plan->cc;
    info[3] = plan->smem_bytes;
    info[4] = plan->var.threads;
    info[5] = plan->nblk;
    info[6] = plan->last_launches;
    info[7] = plan->var.id;
    return DD_OK;
}

dd_status dd_profile_enable(dd_plan plan, int max_executes)
{
    if (!plan)
        return DD_ERR_NULL;
    if (max_executes < 0 || max_executes > (1 << 20))
        return DD_ERR_INVALID_ARG;
    free_prof_events(plan);
    if (max_executes == 0)
        return DD_OK;
    try {
        plan->prof_events.assign(static_cast<size_t>(max_executes) * 3, nullptr);
    } catch (const std::bad_alloc &) {
        return DD_ERR_NOMEM;
    }
    for (void *&e : plan->prof_events) {
        cudaEvent_t ev;
        const cudaError_t ce = cudaEventCreate(&ev);
        if (ce != cudaSuccess) {
            free_prof_events(plan);
            return cuda_fail(ce, "cudaEventCreate");
        }
        e = ev;
    }
    plan->prof_cap = max_executes;
    return DD_OK;
}

dd_status dd_profile_read(dd_plan plan, int *n_executes, float *prepass_ms, float *main_ms)
{
    if (!plan || !n_executes || !prepass_ms || !main_ms)
        return DD_ERR_NULL;
    *n_executes = 0;
    if (plan->prof_cap <= 0)
        return DD_ERR_INVALID_ARG;
    cudaEvent_t *ev = reinterpret_cast<cudaEvent_t *>(plan->prof_events.data());
    const int n = plan->prof_n;
    if (n > 0) {
        cudaError_t ce = cudaEventSynchronize(ev[3 * (n - 1) + 2]);
        if (ce != cudaSuccess)
            return cuda_fail(ce, "cudaEventSynchronize");
        for (int i = 0; i < n; ++i) {
            if ((ce = cudaEventElapsedTime(&prepass_ms[i], ev[3 * i], ev[3 * i + 1])) != cudaSuccess ||
                (ce = cudaEventElapsedTime(&main_ms[i], ev[3 * i + 1], ev[3 * i + 2])) != cudaSuccess)
                return cuda_fail(ce, "cudaEventElapsedTime");
        }
    }
    *n_executes = n;
    plan->prof_n = 0;
    return DD_OK;
}

dd_status dd_int_add_peak(int mode, double *adds_per_sec, void *stream)
{
    if (!adds_per_sec)
        return DD_ERR_NULL;
    if (mode < 0 || mode > 2)
        return DD_ERR_INVALID_ARG;
    const cudaError_t e = int_add_peak(mode, adds_per_sec, static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess)
        return cuda_fail(e, "dd_int_add_peak");
    return DD_OK;
}

const char *dd_strerror(dd_status s)
{
    switch (s) {
    case DD_OK: return "success";
    case DD_ERR_NULL: return "a required pointer is NULL";
    case DD_ERR_INVALID_ARG: return "invalid argument";
    case DD_ERR_NO_DM_LIST: return "no DM list set on this plan";
    case DD_ERR_ALIGNMENT: return "pointer or stride not aligned as required";
    case DD_ERR_STRIDE_TOO_SMALL: return "input rows (or a beam stride) too short for nsamps + max_delay";
    case DD_ERR_OUT_RANGE: return "sums do not fit the requested output type exactly";
    case DD_ERR_DELAY_OVERFLOW: return "a delay does not fit int32";
    case DD_ERR_SMEM: return "delay spread of a DM block does not fit shared memory";
    case DD_ERR_CUDA: return "CUDA error (see dd_last_cuda_error)";
    case DD_ERR_NOMEM: return "host allocation failed";
    case DD_ERR_TOO_LARGE: return "needs more scratch than the static array holds (see dd_last_cuda_error)";
    case DD_ERR_UNSUPPORTED: return "plan not served by this entry point (see dd_last_cuda_error)";
    }
    return "unknown status";
}

const char *dd_last_cuda_error(void) { return g_cuda_error.c_str(); }

}  // extern "C"
