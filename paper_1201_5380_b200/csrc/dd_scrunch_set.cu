// dd_scrunch_set.cu -- the direct transform with time-scrunching (include/dd.h
// "dd_scrunch_*"; readings T1-T4 of DESIGN.md section 11).
//
// Host orchestration only: one ordinary plan per resolution level (created through the C ABI with dt * F), a
// cascade of pair-adding kernels (dd_scrunch.cu) that halves the time resolution stage by stage, and one
// dd_execute per level on the rows of its resolution.  All arithmetic on samples runs in those kernels.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <new>
#include <vector>

#include <cuda_runtime.h>

#include "dd_kernels.cuh"

namespace {

const double kDm = 4.148808e3;   // k_DM in MHz^2 pc^-1 cm^3 s

int64_t ceil16(int64_t x) { return (x + 15) / 16 * 16; }

struct Stage {          // rows at resolution dt * factor (factor >= 2), made from the stage before (or from the input)
    int factor = 1;
    int nbits = 0;      // packed width that holds factor * (2^nbits_in - 1)
    int64_t bytes = 0;  // bytes per row (multiple of 16) for the current nsamps
    uint8_t *rows = nullptr;
};

struct Level {
    int factor = 1, nbits = 0, first = 0, ndm = 0;
    int64_t max_delay = 0;
    dd_plan plan = nullptr;
    int stage = -1;     // index into stages; -1 = the input itself
};

}  // namespace

struct dd_scrunch_s {
    int nchans = 0, nbits = 0;
    double dm_diag = 0;
    std::vector<Stage> stages;
    std::vector<Level> levels;
    int64_t sized_for = -1;   // nsamps the stage buffers were sized for
    int64_t need1 = 0;        // bytes per input row for that nsamps
};

namespace {

// packed width of the series at factor F for nbits_in input: the smallest of 2/4/8 bits holding F * vmax; 0 = none
int width_for(int nbits_in, int factor)
{
    const int64_t top = static_cast<int64_t>(factor) * ((1 << nbits_in) - 1);
    for (int w : {2, 4, 8})
        if (w >= nbits_in && top <= (1 << w) - 1)
            return w;
    return 0;
}

// Sizes of every stage for `nsamps`, backwards from the coarsest: a stage must hold what its own level reads
// (nsamps / F + max delay samples) and the whole 16-byte groups the next stage's pair-adding kernel reads.
int64_t plan_sizes(dd_scrunch_s *s, int64_t nsamps, std::vector<int64_t> *bytes)
{
    const int ns = static_cast<int>(s->stages.size());
    bytes->assign(ns, 0);
    int64_t need_in = 0;   // bytes of the input row
    std::vector<int64_t> own(ns + 1, 0);   // [0] = input, [k + 1] = stage k
    for (const Level &l : s->levels) {
        const int64_t samples = nsamps / l.factor + l.max_delay;
        own[l.stage + 1] = std::max(own[l.stage + 1], ceil16((samples * l.nbits + 7) / 8));
    }
    int64_t next_in = 0;   // bytes the stage after this one reads from this one
    for (int k = ns - 1; k >= 0; --k) {
        (*bytes)[k] = std::max<int64_t>(std::max(own[k + 1], next_in), 16);
        const int nb_prev = k > 0 ? s->stages[k - 1].nbits : s->nbits;
        next_in = (*bytes)[k] * 2 * nb_prev / s->stages[k].nbits;
    }
    need_in = std::max<int64_t>(std::max(own[0], next_in), 16);
    return need_in;
}

}  // namespace

extern "C" {

dd_status dd_scrunch_create(dd_scrunch *set, int nchans, double dt, double f_top, double df, int nbits,
                            const double *dm_list, int ndm, int max_factor)
{
    if (!set || !dm_list)
        return DD_ERR_NULL;
    *set = nullptr;
    if (ndm <= 0 || max_factor < 1 || (max_factor & (max_factor - 1)) != 0)
        return DD_ERR_INVALID_ARG;
    for (int d = 0; d < ndm; ++d)
        if (!(dm_list[d] >= 0.0) || !std::isfinite(dm_list[d]) || (d > 0 && dm_list[d] < dm_list[d - 1]))
            return DD_ERR_INVALID_ARG;
    // a throw-away plan validates the observing parameters
    dd_plan probe = nullptr;
    dd_status st = dd_plan_create(&probe, nchans, dt, f_top, df, nbits);
    if (st != DD_OK)
        return st;
    dd_plan_destroy(probe);

    dd_scrunch_s *s = new (std::nothrow) dd_scrunch_s();
    if (!s)
        return DD_ERR_NOMEM;
    s->nchans = nchans;
    s->nbits = nbits;
    // the diagonal: unit gradient between the last two channels, where the delay is greatest
    if (nchans >= 2) {
        const double fa = f_top + (nchans - 2) * df, fb = f_top + (nchans - 1) * df;
        const double grad = kDm * (1.0 / (fb * fb) - 1.0 / (fa * fa)) / dt;   // samples per unit DM per channel
        s->dm_diag = grad > 0 ? 1.0 / grad : INFINITY;
    } else {
        s->dm_diag = INFINITY;
    }
    // factor per trial (reading T1), capped by max_factor and by the 8-bit packed width
    std::vector<int> factor(ndm, 1);
    for (int d = 0; d < ndm; ++d) {
        int f = 1;
        while (f < max_factor && width_for(nbits, 2 * f) != 0 && dm_list[d] > s->dm_diag * (2.0 * f))
            f *= 2;
        factor[d] = f;
    }
    const int fmax = factor[ndm - 1];   // non-decreasing list -> non-decreasing factors
    for (int f = 2; f <= fmax; f *= 2) {
        Stage sg;
        sg.factor = f;
        sg.nbits = width_for(nbits, f);
        s->stages.push_back(sg);
    }
    for (int d = 0; d < ndm;) {
        int e = d;
        while (e < ndm && factor[e] == factor[d])
            ++e;
        Level l;
        l.factor = factor[d];
        l.nbits = width_for(nbits, l.factor);
        l.first = d;
        l.ndm = e - d;
        l.stage = -1;
        for (size_t k = 0; k < s->stages.size(); ++k)
            if (s->stages[k].factor == l.factor)
                l.stage = static_cast<int>(k);
        st = dd_plan_create(&l.plan, nchans, dt * l.factor, f_top, df, l.nbits);
        if (st == DD_OK && l.factor > 1)   // a sample of the series at F dt is at most F (2^nbits - 1)
            st = dd_set_input_max(l.plan, l.factor * ((1 << nbits) - 1));
        if (st == DD_OK)
            st = dd_set_dm_list(l.plan, dm_list + d, l.ndm);
        if (st == DD_OK) {
            l.max_delay = dd_get_max_delay(l.plan);
            s->levels.push_back(l);
        } else {
            if (l.plan)
                dd_plan_destroy(l.plan);
            dd_scrunch_destroy(s);
            return st;
        }
        d = e;
    }
    *set = s;
    return DD_OK;
}

dd_status dd_scrunch_set_killmask(dd_scrunch set, const int32_t *mask)
{
    if (!set)
        return DD_ERR_NULL;
    for (Level &l : set->levels) {   // the same channels are left out at every resolution
        const dd_status st = dd_set_killmask(l.plan, mask);
        if (st != DD_OK)
            return st;
    }
    return DD_OK;
}

int dd_scrunch_levels(dd_scrunch set) { return set ? static_cast<int>(set->levels.size()) : DD_ERR_NULL; }

dd_status dd_scrunch_level_info(dd_scrunch set, int level, int64_t *info)
{
    if (!set || !info)
        return DD_ERR_NULL;
    if (level < 0 || level >= static_cast<int>(set->levels.size()))
        return DD_ERR_INVALID_ARG;
    const Level &l = set->levels[level];
    info[0] = l.factor;
    info[1] = l.first;
    info[2] = l.ndm;
    info[3] = l.max_delay;
    info[4] = l.nbits;
    info[5] = std::isfinite(set->dm_diag) ? static_cast<int64_t>(std::llround(set->dm_diag * 1e6)) : -1;
    return DD_OK;
}

int64_t dd_scrunch_required_bytes(dd_scrunch set, int64_t nsamps)
{
    if (!set)
        return DD_ERR_NULL;
    if (nsamps < set->levels.back().factor || nsamps > (INT64_MAX >> 8))
        return DD_ERR_INVALID_ARG;
    std::vector<int64_t> bytes;
    return plan_sizes(set, nsamps, &bytes);
}

dd_status dd_scrunch_execute(dd_scrunch set, int64_t nsamps, const void *in_ptr, int64_t in_stride, void *const *out_ptrs,
                             int out_nbits, void *stream)
{
    if (!set || !in_ptr || !out_ptrs)
        return DD_ERR_NULL;
    if (nsamps < set->levels.back().factor || nsamps > (INT64_MAX >> 8))
        return DD_ERR_INVALID_ARG;
    if (reinterpret_cast<uintptr_t>(in_ptr) % 16 != 0 || in_stride <= 0 || in_stride % 16 != 0)
        return DD_ERR_ALIGNMENT;
    for (size_t l = 0; l < set->levels.size(); ++l)
        if (!out_ptrs[l])
            return DD_ERR_NULL;
    std::vector<int64_t> bytes;
    const int64_t need_in = plan_sizes(set, nsamps, &bytes);
    if (in_stride < need_in)
        return DD_ERR_STRIDE_TOO_SMALL;
    cudaStream_t st_ = static_cast<cudaStream_t>(stream);
    if (set->sized_for != nsamps) {
        for (size_t k = 0; k < set->stages.size(); ++k) {
            Stage &sg = set->stages[k];
            if (sg.bytes < bytes[k] || !sg.rows) {
                if (sg.rows)
                    cudaFree(sg.rows);   // synchronises with kernels still using the old rows
                sg.rows = nullptr;
                if (cudaMalloc(&sg.rows, static_cast<size_t>(bytes[k]) * set->nchans) != cudaSuccess) {
                    (void)cudaGetLastError();
                    set->sized_for = -1;
                    return DD_ERR_NOMEM;
                }
            }
            sg.bytes = bytes[k];
        }
        set->sized_for = nsamps;
        set->need1 = need_in;
    }
    // the cascade: every stage adds adjacent pairs of the one before
    const uint8_t *src = static_cast<const uint8_t *>(in_ptr);
    int64_t src_stride = in_stride;
    int src_bits = set->nbits;
    for (Stage &sg : set->stages) {
        const cudaError_t e = dd::launch_scrunch(src_bits, sg.nbits, set->nchans, src, src_stride, sg.rows, sg.bytes, sg.bytes, st_);
        if (e != cudaSuccess) {
            (void)cudaGetLastError();
            return DD_ERR_CUDA;
        }
        src = sg.rows;
        src_stride = sg.bytes;
        src_bits = sg.nbits;
    }
    for (size_t l = 0; l < set->levels.size(); ++l) {
        const Level &lv = set->levels[l];
        const void *rows = lv.stage < 0 ? in_ptr : set->stages[lv.stage].rows;
        const int64_t stride = lv.stage < 0 ? in_stride : set->stages[lv.stage].bytes;
        const dd_status st = dd_execute(lv.plan, nsamps / lv.factor, rows, stride, out_ptrs[l], out_nbits, stream);
        if (st != DD_OK)
            return st;
    }
    return DD_OK;
}

dd_status dd_scrunch_destroy(dd_scrunch set)
{
    if (!set)
        return DD_ERR_NULL;
    for (Level &l : set->levels)
        if (l.plan)
            dd_plan_destroy(l.plan);
    for (Stage &sg : set->stages)
        if (sg.rows)
            cudaFree(sg.rows);
    delete set;
    return DD_OK;
}

}  // extern "C"
