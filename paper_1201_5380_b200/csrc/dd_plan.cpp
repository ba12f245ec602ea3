// dd_plan.cpp -- host-side planning: the delay table (double precision) and the tile metadata.
#include "dd_plan.h"

#include <algorithm>
#include <cmath>
#include <limits>

namespace dd {

// Dispersion constant k_DM in MHz^2 pc^-1 cm^3 s.
static const double kDispersionConstant = 4.148808e3;

// eq. 4-5 in double precision on the host; "rounded to the nearest integer"
// is taken as floor(x + 0.5) (reading R1; x >= 0 for a descending band).
dd_status compute_delay_table(dd_plan_s *p)
{
    const int nchans = p->nchans, ndm = p->ndm;
    std::vector<double> band(nchans);   // f_c^-2 - f_top^-2, shared by all DM trials
    const double inv_top2 = 1.0 / (p->f_top * p->f_top);
    for (int c = 0; c < nchans; ++c) {
        const double f = p->f_top + static_cast<double>(c) * p->df;
        band[c] = 1.0 / (f * f) - inv_top2;
    }
    std::vector<int32_t> table(static_cast<size_t>(ndm) * nchans);
    int64_t maxd = 0;
    for (int d = 0; d < ndm; ++d) {
        const double scale = kDispersionConstant * p->dm[d];
        int32_t *row = table.data() + static_cast<size_t>(d) * nchans;
        for (int c = 0; c < nchans; ++c) {
            const double x = scale * band[c] / p->dt;
            const double r = std::floor(x + 0.5);
            if (!(r >= 0.0) || r > static_cast<double>(std::numeric_limits<int32_t>::max() - 1))
                return DD_ERR_DELAY_OVERFLOW;
            row[c] = static_cast<int32_t>(r);
            maxd = std::max<int64_t>(maxd, row[c]);
        }
    }
    p->delay.swap(table);
    p->max_delay = maxd;
    return DD_OK;
}

static inline int64_t align_up(int64_t x, int64_t a) { return (x + a - 1) / a * a; }

// Sub-band method: "the direct dedispersion algorithm is applied to sub-bands of N'nu channels
// to compute a dedispersed time series for each nominal DM and sub-band.  In the second step, the DM trials near
// each nominal value are computed by applying the direct algorithm to the miniature filterbanks".  Readings
// S1-S4 of DESIGN.md section 10: groups of dm_group consecutive trials, nominal = the group's middle trial;
// step-1 delays by eq. 4-5 relative to the sub-band's first channel; step-2 delays = the full-band delays of
// the sub-bands' first channels.
dd_status build_subband(const dd_plan_s *p, dd_plan_s *s1, dd_plan_s *s2, std::vector<int32_t> *nominal,
                        int64_t *max_d2, int64_t *extent)
{
    const int nchans = p->nchans, ndm = p->ndm, sb = p->sb_nchans, grp = p->dm_group;
    const int nsb = nchans / sb, ngrp = (ndm + grp - 1) / grp;
    nominal->resize(ngrp);
    for (int g = 0; g < ngrp; ++g)
        (*nominal)[g] = std::min(g * grp + grp / 2, ndm - 1);
    // step 1: nominal DMs, every channel delayed relative to the first channel of its sub-band
    s1->nchans = nchans;
    s1->dt = p->dt;
    s1->f_top = p->f_top;
    s1->df = p->df;
    s1->nbits = p->nbits;
    s1->ndm = ngrp;
    s1->dm.resize(ngrp);
    s1->keep = p->keep;
    s1->group_size = sb;
    s1->force_variant = 3;
    s1->delay.resize(static_cast<size_t>(ngrp) * nchans);
    std::vector<double> band(nchans);
    for (int c = 0; c < nchans; ++c) {
        const double f = p->f_top + static_cast<double>(c) * p->df;
        const double f_sb = p->f_top + static_cast<double>(c / sb * sb) * p->df;
        band[c] = 1.0 / (f * f) - 1.0 / (f_sb * f_sb);
    }
    std::vector<int64_t> d1max(nsb, 0);
    int64_t maxd = 0;
    for (int g = 0; g < ngrp; ++g) {
        s1->dm[g] = p->dm[(*nominal)[g]];
        const double scale = kDispersionConstant * s1->dm[g];
        for (int c = 0; c < nchans; ++c) {
            const double r = std::floor(scale * band[c] / p->dt + 0.5);
            if (!(r >= 0.0) || r > static_cast<double>(std::numeric_limits<int32_t>::max() - 1))
                return DD_ERR_DELAY_OVERFLOW;
            const int32_t v = static_cast<int32_t>(r);
            s1->delay[static_cast<size_t>(g) * nchans + c] = v;
            d1max[c / sb] = std::max<int64_t>(d1max[c / sb], v);
            maxd = std::max<int64_t>(maxd, v);
        }
    }
    s1->max_delay = maxd;
    // step 2: N_SB channels at the sub-bands' first frequencies, all trials, delays taken from the full table
    s2->nchans = nsb;
    s2->dt = p->dt;
    s2->f_top = p->f_top;
    s2->df = p->df * sb;
    s2->nbits = 8;
    s2->ndm = ndm;
    s2->dm = p->dm;
    s2->force_variant = 3;
    {   // the largest sample of the miniature filterbanks: live channels of the fullest sub-band times the largest input
        int most = 0;
        for (int b = 0; b < nsb; ++b) {
            int n = 0;
            for (int c = b * sb; c < (b + 1) * sb; ++c)
                n += (p->keep.empty() || p->keep[c]) ? 1 : 0;
            most = std::max(most, n);
        }
        int64_t vtop = static_cast<int64_t>(most) * ((1 << p->nbits) - 1);
        s2->in_planes = 1;
        while ((int64_t(1) << s2->in_planes) <= vtop)
            ++s2->in_planes;
    }
    s2->delay.resize(static_cast<size_t>(ndm) * nsb);
    int64_t m2 = 0, ext = 0;
    for (int b = 0; b < nsb; ++b) {
        int64_t colmax = 0;
        for (int d = 0; d < ndm; ++d) {
            const int32_t v = p->delay[static_cast<size_t>(d) * nchans + static_cast<size_t>(b) * sb];
            s2->delay[static_cast<size_t>(d) * nsb + b] = v;
            colmax = std::max<int64_t>(colmax, v);
        }
        m2 = std::max(m2, colmax);
        ext = std::max(ext, colmax + d1max[b]);
    }
    s2->max_delay = m2;
    *max_d2 = m2;
    *extent = ext;
    dd_status st = build_tiles(s1);
    if (st != DD_OK)
        return st;
    return build_tiles(s2);
}

int64_t smem_layout_bytes(const dd_plan_s *p, int cc)
{
    const Variant &v = p->var;
    int64_t bytes = 128;                                                                          // mbarriers
    if (p->patch)   // one output patch per warp for the coalescing epilogue (kept apart from the stages,
        bytes += static_cast<int64_t>(v.threads / 32) * kBpPatchBytes;   // so that a warp can store while others still add); Bp<nbits>::PATCH
    bytes += p->nstages * align_up(static_cast<int64_t>(cc) * v.DB * v.rel_bytes, 128);           // offset-table stages
    bytes += p->nstages * align_up(static_cast<int64_t>(p->pairs ? p->rows_per_chunk : cc) * p->raw_slot, 128);   // packed / bit-plane stages (pair rows: rows per stage)
    if (v.lane_bits != p->nbits)                                                                  // unpacked lanes
        bytes += v.lane_stages * align_up(static_cast<int64_t>(cc) * p->lane_slot, 128);
    return bytes;
}

// Stages between flushes in the LONG bit-plane kernel: must agree with Bp<nbits>::FL (DD_BP_FL*) in dd_kernel_bp.cu.
#ifndef DD_PAIR_FL
#define DD_PAIR_FL 4
#endif
#ifndef DD_BP_W2
#define DD_BP_W2 5
#endif
#ifndef DD_BP_FL2
#define DD_BP_FL2 2
#define DD_BP_FL4 4
#define DD_BP_FL8 2
#endif
static int kBpFlushStages(int nbits) { return nbits == 2 ? DD_BP_FL2 : (nbits == 4 ? DD_BP_FL4 : DD_BP_FL8); }

// The kernel variants compiled into the library, in order of preference.
static const Variant kVariants[] = {
    /* id  DB   TB    thr tail rel lane lst rst  cc candidates     nbits                        sum  pad    bitplane */
    // bit planes + carry-save counters (dd_kernel_bp.cu): tile shapes must match Bp<nbits> there
    {3, 16, 1024 * DD_BP_W2, 512, 32, 8, 2, 0, 4, {32, 0, 0, 0}, 1 << 2, 12, true, true, 8, 1},      // 2-bit: 2 planes, W = 5
    {3, 16, 3072, 512, 32, 8, 4, 0, 4, {16, 0, 0, 0}, 1 << 4, 16, true, true, 16, 1},              // 4-bit: 4 planes, W = 3
    {3, 16, 3072, 512, 32, 8, 8, 0, 4, {8, 0, 0, 0}, 1 << 8, 20, true, true, 16, 2},               // 8-bit: 2 x 4 planes, W = 3
    {2, 32, 1280, 512, 8, 4, 4, 2, 2, {40, 20, 10, 5}, 1 << 2, 16, false, false, 0, 1},            // 2-bit, nibble lanes
    {1, 32, 640, 256, 4, 2, 8, 1, 2, {32, 16, 8, 4}, (1 << 2) | (1 << 4) | (1 << 8), 32, false, false, 0, 1},
};

// Variant 4 -- pair rows.  For two adjacent live channels (c0, c1) the difference delta = delay[d][c1] - delay[d][c0]
// takes few values over the whole DM list (it grows slowly with DM and the two roundings make it jitter by one), so
// the row S_delta[t] = x[c0][t] + x[c1][t + delta] is made ONCE per delta by a pre-pass (n + 1 bit planes), and every
// trial adds the row of its own delta at the delay of c0: n + 1 plane words per pair instead of 2 n.  Exact: the
// delay table is used as it stands.  The transform kernel is the bit-plane kernel of the next width (2-bit pairs:
// the 4-plane layout with 3 planes in use; 4-bit pairs: the 2 x 4-plane layout with 5 in use); a stage holds CC
// pairs and the rows of every delta the DM block needs for them.
dd_status build_tiles_pairs(dd_plan_s *p)
{
    const int nrows = p->nchans, ndm = p->ndm, nbits = p->nbits;
    if (p->group_size > 0)
        return DD_ERR_SMEM;
    std::vector<int32_t> live;
    for (int c = 0; c < nrows; ++c)
        if (p->keep.empty() || p->keep[c])
            live.push_back(c);
    const int nlive = static_cast<int>(live.size());
    if (nlive == 0)
        return DD_ERR_SMEM;
    const int npairs = (nlive + 1) / 2;
    const int enb = nbits == 2 ? 3 : (nbits == 4 ? 8 : 12);   // layout of the pair rows (must match Bp<3> / Bp<8> / Bp<12> in dd_kernel_bp.cu)
    Variant v{};
    if (nbits == 2) {   // 3 planes per unit (12 bytes), 5 units per lane, 8 pairs per stage, flush every 4 stages
        v = Variant{4, 16, 1024 * DD_BP_W2, 512, 32, 8, 3, 0, 4, {8, 0, 0, 0}, 1 << 2, 12, true, true, 12, 1};
    } else if (nbits == 8) {   // 9 planes in three 4-plane sub-rows, 3 units per lane, 4 pairs per stage, flush every 2 stages
        v = Variant{4, 16, 3072, 512, 32, 8, 12, 0, 4, {4, 0, 0, 0}, 1 << 8, 20, true, true, 16, 3};
    } else {
        const Variant *vv = nullptr;
        for (const Variant &k : kVariants)
            if (k.id == 3 && (k.nbits_mask & (1 << enb)))
                vv = &k;
        if (!vv)
            return DD_ERR_SMEM;
        v = *vv;
        v.id = 4;
    }
    const int pin = nbits + 1;                          // planes of a pair sum
    const int64_t top = static_cast<int64_t>(npairs) * ((1 << pin) - 1);   // structural weight the counters take
    if (top >= (int64_t(1) << (nbits == 4 ? 16 : v.max_sum_bits)))   // 4-bit pairs: the kernel keeps 16 sum planes
        return DD_ERR_SMEM;
    const int DB = v.DB, cc = v.cc[0];
    const int fl = DD_PAIR_FL;   // stages between flushes of the pair-row kernels (dd_kernel_bp.cu: the same)
    const int nblk = (ndm + DB - 1) / DB;
    const bool long_mode = npairs >= 8 * cc * fl;
    const int ents_pad = static_cast<int>(align_up(npairs, cc * (long_mode ? fl : 1)));
    const int nchunks = ents_pad / cc;
    // pair rows: every delta of every pair, in pair order
    std::vector<int32_t> prow;
    std::vector<int64_t> rowbase(npairs + 1, 0);
    std::vector<std::vector<int32_t>> deltas(npairs);
    for (int q = 0; q < npairs; ++q) {
        const int c0 = live[2 * q], c1 = 2 * q + 1 < nlive ? live[2 * q + 1] : -1;
        std::vector<int32_t> &u = deltas[q];
        if (c1 < 0) {
            u.push_back(0);
        } else {
            for (int d = 0; d < ndm; ++d)
                u.push_back(p->delay[static_cast<size_t>(d) * nrows + c1] - p->delay[static_cast<size_t>(d) * nrows + c0]);
            std::sort(u.begin(), u.end());
            u.erase(std::unique(u.begin(), u.end()), u.end());
        }
        rowbase[q + 1] = rowbase[q] + static_cast<int64_t>(u.size());
        for (int32_t dl : u) {
            prow.push_back(c0);
            prow.push_back(c1);
            prow.push_back(dl);
            prow.push_back(0);
        }
    }
    const int64_t n_prows = rowbase[npairs];
    if (n_prows > (int64_t(1) << 30))
        return DD_ERR_SMEM;
    // per (DM block, pair): the rows in use and the staged span (of the pair's first channel)
    const bool lone = nbits != 2;   // last sub-row of a pair row: the carry plane alone, 4 bytes per unit (dd_kernel_bp.cu LONE)
    const int A = 128;              // spans in whole groups of 4 units: 12-byte units and quarter-size lone sub-rows stay 16-byte aligned
    struct Use { int32_t start, nbytes; std::vector<int32_t> rows; };
    std::vector<Use> use(static_cast<size_t>(nblk) * npairs);
    int64_t max_bytes = 0, max_end = 0;
    int rs = 0;
    for (int b = 0; b < nblk; ++b) {
        for (int k = 0; k < nchunks; ++k) {
            int rows_here = 0;
            for (int e = k * cc; e < std::min((k + 1) * cc, npairs); ++e) {
                const int c0 = live[2 * e], c1 = 2 * e + 1 < nlive ? live[2 * e + 1] : -1;
                int32_t dmin = std::numeric_limits<int32_t>::max(), dmax = 0;
                Use &u = use[static_cast<size_t>(b) * npairs + e];
                for (int i = 0; i < DB; ++i) {
                    const int d = std::min(b * DB + i, ndm - 1);
                    const int32_t d0 = p->delay[static_cast<size_t>(d) * nrows + c0];
                    const int32_t dl = c1 < 0 ? 0 : p->delay[static_cast<size_t>(d) * nrows + c1] - d0;
                    dmin = std::min(dmin, d0);
                    dmax = std::max(dmax, d0);
                    const int32_t r = static_cast<int32_t>(
                        rowbase[e] + (std::lower_bound(deltas[e].begin(), deltas[e].end(), dl) - deltas[e].begin()));
                    if (std::find(u.rows.begin(), u.rows.end(), r) == u.rows.end())
                        u.rows.push_back(r);
                }
                const int32_t start = dmin / A * A;
                const int64_t need = static_cast<int64_t>(v.TB) + (dmax - start) + v.tail;
                const int64_t nbytes = align_up(need, A) / 32 * v.unit_bytes;
                if (dmax - start > (int64_t(1) << 26) || nbytes > (1 << 19))
                    return DD_ERR_SMEM;
                u.start = start;
                u.nbytes = static_cast<int32_t>(nbytes);
                max_bytes = std::max(max_bytes, nbytes);
                max_end = std::max<int64_t>(max_end, start + nbytes / v.unit_bytes * 32);
                rows_here += static_cast<int>(u.rows.size());
            }
            if ((k + 1) * cc > npairs)
                rows_here += 1;   // the all-zero row behind which the padded entries of this stage hide
            rs = std::max(rs, rows_here);
        }
    }
    rs = std::max(rs, 1);
    if (rs > 48)   // the kernel's producers stage at most 3 rows per warp and stage
        return DD_ERR_SMEM;
    p->var = v;
    p->pairs = true;
    p->pair_nbits = enb;
    p->pair_planes = pin;
    p->long_mode = long_mode;
    p->patch = !long_mode || nbits == 2;   // 4- and 8-bit input, long: no output patches, a deeper ring (must match PATCH in dd_kernel_bp.cu)
    p->max_span_end = max_end;
    p->sub_slot = static_cast<int>(max_bytes);
    p->raw_slot = lone ? static_cast<int>(max_bytes) * (v.nsub - 1) + static_cast<int>(max_bytes) / 4 : static_cast<int>(max_bytes) * v.nsub;
    p->lane_slot = p->raw_slot;
    p->rows_per_chunk = rs;
    p->cc = cc;
    int nst = 0;
    for (int n = v.raw_stages; n >= 2 && nst == 0; --n) {
        p->nstages = n;
        const int64_t tx = static_cast<int64_t>(rs) * p->raw_slot + static_cast<int64_t>(cc) * DB * v.rel_bytes;
        if (smem_layout_bytes(p, cc) <= kMaxDynSmem && tx < (1 << 20))
            nst = n;
    }
    if (nst == 0) {
        p->pairs = false;
        return DD_ERR_SMEM;
    }
    p->nstages = nst;
    // span list [nblk][nchunks][rs] and offsets [nblk][ents_pad][DB]
    std::vector<SpanMeta> span(static_cast<size_t>(nblk) * nchunks * rs);
    std::vector<uint8_t> rel(static_cast<size_t>(nblk) * ents_pad * DB * 8);
    for (int b = 0; b < nblk; ++b) {
        for (int k = 0; k < nchunks; ++k) {
            SpanMeta *sl = span.data() + (static_cast<size_t>(b) * nchunks + k) * rs;
            int slot = 0;
            for (int j = 0; j < rs; ++j)
                sl[j] = SpanMeta{0, 0, 0, 0};
            int zero_slot = -1;   // a stage with padded entries also stages the all-zero row (row n_prows)
            for (int e = k * cc; e < (k + 1) * cc; ++e) {
                const size_t base = (static_cast<size_t>(b) * ents_pad + e) * DB;
                if (e >= npairs) {   // padded entry: every window at the start of the zero row's slot
                    if (zero_slot < 0) {
                        zero_slot = slot;
                        sl[slot] = SpanMeta{0, p->sub_slot, static_cast<int32_t>(n_prows), 0};
                        ++slot;
                    }
                    for (int i = 0; i < DB; ++i) {
                        uint32_t *en = reinterpret_cast<uint32_t *>(rel.data()) + (base + i) * 2;
                        en[0] = static_cast<uint32_t>(zero_slot) * static_cast<uint32_t>(p->raw_slot);
                        en[1] = 0;
                    }
                    continue;
                }
                const Use &u = use[static_cast<size_t>(b) * npairs + e];
                const int first_slot = slot;
                for (int32_t r : u.rows) {
                    sl[slot] = SpanMeta{u.start / 32 * v.unit_bytes, u.nbytes, r, u.start};
                    ++slot;
                }
                const int c0 = live[2 * e], c1 = 2 * e + 1 < nlive ? live[2 * e + 1] : -1;
                for (int i = 0; i < DB; ++i) {
                    const int d = std::min(b * DB + i, ndm - 1);
                    const int32_t d0 = p->delay[static_cast<size_t>(d) * nrows + c0];
                    const int32_t dl = c1 < 0 ? 0 : p->delay[static_cast<size_t>(d) * nrows + c1] - d0;
                    const int32_t r = static_cast<int32_t>(
                        rowbase[e] + (std::lower_bound(deltas[e].begin(), deltas[e].end(), dl) - deltas[e].begin()));
                    const int which = static_cast<int>(std::find(u.rows.begin(), u.rows.end(), r) - u.rows.begin());
                    const uint32_t off = static_cast<uint32_t>(d0 - u.start);
                    uint32_t *en = reinterpret_cast<uint32_t *>(rel.data()) + (base + i) * 2;
                    en[0] = static_cast<uint32_t>(first_slot + which) * static_cast<uint32_t>(p->raw_slot) +
                            (off >> 5) * static_cast<uint32_t>(v.unit_bytes);
                    en[1] = (off & 31u) | ((off >> 5) << 8);   // shift; unit offset for the lone sub-row
                }
            }
        }
    }
    p->ngroups = 1;
    p->group_cols = ents_pad;
    p->nblk = nblk;
    p->nchans_pad = ents_pad;
    p->smem_bytes = smem_layout_bytes(p, cc);
    p->span.swap(span);
    p->rel.swap(rel);
    p->live.swap(live);
    p->nlive = nlive;
    p->prow.swap(prow);
    p->n_prows = n_prows;
    const int64_t vmax = (1 << nbits) - 1;
    p->final32 = static_cast<int64_t>(nlive) * vmax > 65535;
    return DD_OK;
}

int64_t gs_smem_bytes(int nbits, int G, int cc, int rows, int row_units, int raw_sub, int nsr, int nsp, bool patch)
{
    const int nsubr = nbits == 8 ? 2 : 1, pin = nbits + (G == 2 ? 1 : 2);
    int64_t b = 128 + (patch ? 16 * static_cast<int64_t>(kBpPatchBytes) : 0);
    b += nsp * align_up(static_cast<int64_t>(cc) * 16 * 8, 128);                       // offset entries of the trials
    b += nsr * align_up(static_cast<int64_t>(rows) * 64, 128);                         // build table
    b += nsr * align_up(static_cast<int64_t>(G) * cc * nsubr * raw_sub, 128);          // staged bit-plane spans
    b += nsp * align_up(static_cast<int64_t>(rows) * row_units * 4 * pin, 128);        // rows
    return b;
}

// Variant 5 -- group sums made inside the CTA (dd_kernel_gs.cu).  Groups of G adjacent live channels; per (DM block,
// group) the distinct patterns (delta_1 .. delta_{G-1}), delta_i = delay[d][c_i] - delay[d][c_0], of the block's 16
// trials; the CTA builds one row R[t] = sum_i x[c_i][t + delta_i] per pattern from the staged spans of the G channels
// and every trial adds the row of its own pattern at the delay of c_0.  Exact: the delay table is used as it stands.
dd_status build_tiles_gs(dd_plan_s *p, int G, int cc)
{
    const int nrows = p->nchans, ndm = p->ndm, nbits = p->nbits;
    if (p->group_size > 0 || p->in_planes > 0 || (G != 2 && G != 4) || !gs_instance_exists(nbits, G, cc))
        return DD_ERR_SMEM;
    std::vector<int32_t> live;
    for (int c = 0; c < nrows; ++c)
        if (p->keep.empty() || p->keep[c])
            live.push_back(c);
    const int nlive = static_cast<int>(live.size());
    if (nlive == 0)
        return DD_ERR_SMEM;
    const int W = nbits == 2 ? kGsW2 : kGsW48, TB = 1024 * W, DB = 16;
    const int nbr = nbits == 2 ? 2 : 4, nsubr = nbits / nbr, ubr = nbr * 4;   // raw layout: planes per unit, sub-rows, bytes per unit
    const int pin = nbits + (G == 2 ? 1 : 2), np = nbits == 2 ? 12 : (nbits == 4 ? 16 : 20);
    const int64_t vmax = (1 << nbits) - 1;
    if (static_cast<int64_t>(nlive) * vmax >= (int64_t(1) << np))
        return DD_ERR_SMEM;
    const int ngr = (nlive + G - 1) / G, fl = kGsFlushStages;
    const int ents_pad = static_cast<int>(align_up(ngr, cc * fl)), nchunks = ents_pad / cc;
    const int nblk = (ndm + DB - 1) / DB;
    const int A = 32 * (16 / ubr);   // samples per 16 bytes of a raw sub-row: the bulk-copy granularity

    struct GInfo {
        int cnt = 0;                 // channels present
        int32_t ch[4] = {0, 0, 0, 0};
        int32_t start0 = 0, U = 0;   // first sample of the rows (multiple of 32), units per row
        int npat = 0;
        int32_t pat[16][4];          // delay differences per pattern
        uint8_t pat_of[16];          // pattern of every trial
        int32_t off[16];             // delay[d][c_0] - start0
        int32_t rawstart[4], RU[4];  // staged span per channel: first sample, units
    };
    auto analyse = [&](int b, int q, GInfo &g) -> bool {
        g = GInfo();
        if (q >= ngr) {   // padded group: one all-zero row
            g.U = TB / 32 + 1;
            g.npat = 1;
            for (int i = 0; i < 4; ++i)
                g.pat[0][i] = 0, g.rawstart[i] = 0, g.RU[i] = 0;
            for (int i = 0; i < DB; ++i)
                g.pat_of[i] = 0, g.off[i] = 0;
            return true;
        }
        g.cnt = std::min(G, nlive - q * G);
        for (int i = 0; i < g.cnt; ++i)
            g.ch[i] = live[q * G + i];
        int32_t dmin = std::numeric_limits<int32_t>::max(), dmax = 0, d0s[16];
        for (int i = 0; i < DB; ++i) {
            const int d = std::min(b * DB + i, ndm - 1);   // the last block is padded with its last trial
            const int32_t *row = p->delay.data() + static_cast<size_t>(d) * nrows;
            d0s[i] = row[g.ch[0]];
            dmin = std::min(dmin, d0s[i]);
            dmax = std::max(dmax, d0s[i]);
            int32_t dl[4] = {0, 0, 0, 0};
            for (int k = 1; k < g.cnt; ++k)
                dl[k] = row[g.ch[k]] - d0s[i];
            int f = -1;
            for (int k = 0; k < g.npat && f < 0; ++k)
                if (std::equal(dl, dl + 4, g.pat[k]))
                    f = k;
            if (f < 0) {
                f = g.npat++;
                std::copy(dl, dl + 4, g.pat[f]);
            }
            g.pat_of[i] = static_cast<uint8_t>(f);
        }
        g.start0 = dmin / 32 * 32;
        if (dmax - g.start0 > (1 << 20))
            return false;
        g.U = TB / 32 + (dmax - g.start0) / 32 + 1;
        for (int i = 0; i < DB; ++i)
            g.off[i] = d0s[i] - g.start0;
        for (int k = 0; k < g.cnt; ++k) {
            int32_t lo = std::numeric_limits<int32_t>::max(), hi = std::numeric_limits<int32_t>::min();
            for (int j = 0; j < g.npat; ++j) {
                lo = std::min(lo, g.pat[j][k]);
                hi = std::max(hi, g.pat[j][k]);
            }
            if (g.start0 + lo < 0 || hi - lo > (1 << 20))   // (a difference can be negative only in a table that is not
                return false;                                //  monotone in c, i.e. never for df < 0; refused all the same)
            g.rawstart[k] = (g.start0 + lo) / A * A;
            const int ru = ((g.start0 + hi - g.rawstart[k]) >> 5) + g.U + 1;   // the funnel shift reads one unit further
            g.RU[k] = static_cast<int32_t>(align_up(ru, 16 / ubr));
        }
        return true;
    };

    // pass 1: sizes
    int rows = 1, row_units = 0, raw_units = 16 / ubr;
    int64_t max_end = 0;
    GInfo g;
    for (int b = 0; b < nblk; ++b) {
        for (int k = 0; k < nchunks; ++k) {
            int rows_here = 0;
            for (int q = k * cc; q < (k + 1) * cc; ++q) {
                if (!analyse(b, q, g))
                    return DD_ERR_SMEM;
                rows_here += g.npat;
                row_units = std::max(row_units, g.U);
                for (int i = 0; i < g.cnt; ++i) {
                    raw_units = std::max(raw_units, g.RU[i]);
                    max_end = std::max<int64_t>(max_end, static_cast<int64_t>(g.rawstart[i]) + static_cast<int64_t>(g.RU[i]) * 32);
                }
            }
            rows = std::max(rows, rows_here);
        }
    }
    row_units = static_cast<int>(align_up(row_units, 8));   // (two arrays of whole 16-byte groups when W is even)
    if (row_units >= 2048)
        return DD_ERR_SMEM;                                 // unit positions travel in 12 bits
    const int raw_sub = raw_units * ubr;
    max_end = std::max<int64_t>(max_end, static_cast<int64_t>(raw_units) * 32);   // zero-row copies of padded channels
    if (static_cast<int64_t>(rows) * ((row_units + 31) / 32) >= 4096 || raw_sub > (1 << 19))
        return DD_ERR_SMEM;
    // ring depths: the deepest that fits; output patches for 2- and 4-bit input when there is room for them
    const bool want_patch = nbits < 8;
    const int cand[6][3] = {{3, 3, 1}, {2, 3, 1}, {3, 3, 0}, {2, 3, 0}, {2, 2, 1}, {2, 2, 0}};
    int nsr = 0, nsp = 0;
    bool patch = false;
    for (const auto &cd : cand) {
        if (cd[2] && !want_patch)
            continue;
        if (gs_smem_bytes(nbits, G, cc, rows, row_units, raw_sub, cd[0], cd[1], cd[2] != 0) <= kMaxDynSmem) {
            nsr = cd[0], nsp = cd[1], patch = cd[2] != 0;
            break;
        }
    }
    if (nsr == 0)
        return DD_ERR_SMEM;

    // pass 2: tables
    const int CHS = G * cc, row_bytes = row_units * 4 * pin;
    std::vector<SpanMeta> span(static_cast<size_t>(nblk) * nchunks * CHS);
    std::vector<GsEntry> tab(static_cast<size_t>(nblk) * nchunks * rows);
    std::vector<uint8_t> rel(static_cast<size_t>(nblk) * nchunks * cc * DB * 8);
    for (int b = 0; b < nblk; ++b) {
        for (int k = 0; k < nchunks; ++k) {
            const size_t st = static_cast<size_t>(b) * nchunks + k;
            GsEntry *te = tab.data() + st * rows;
            for (int r = 0; r < rows; ++r)
                te[r] = GsEntry{};
            te[0].nunits = 1;   // (entry 0 is always in use; guards the builder's clamp if it were not)
            int row_idx = 0;
            for (int gi = 0; gi < cc; ++gi) {
                analyse(b, k * cc + gi, g);
                for (int i = 0; i < G; ++i) {
                    SpanMeta &m = span[st * CHS + gi * G + i];
                    if (i < g.cnt)
                        m = SpanMeta{g.rawstart[i] / 32 * ubr, g.RU[i] * ubr, g.ch[i], 0};
                    else
                        m = SpanMeta{0, raw_sub, nrows, 0};   // the all-zero row behind the input rows
                }
                for (int j = 0; j < g.npat; ++j) {
                    GsEntry &e = te[row_idx + j];
                    e.dst = (row_idx + j) * row_bytes;
                    e.nunits = g.U;
                    for (int i = 0; i < G; ++i) {
                        const int32_t o = i < g.cnt ? g.start0 + g.pat[j][i] - g.rawstart[i] : 0;
                        e.src[i] = (gi * G + i) * nsubr * raw_sub + (o >> 5) * ubr;
                        e.sh[i] = o & 31;
                    }
                }
                uint32_t *en = reinterpret_cast<uint32_t *>(rel.data()) + (st * cc + gi) * DB * 2;
                for (int i = 0; i < DB; ++i) {
                    const uint32_t off = static_cast<uint32_t>(g.off[i]);
                    en[2 * i] = static_cast<uint32_t>(row_idx + g.pat_of[i]) * static_cast<uint32_t>(row_bytes);
                    // positions of the trial's first and second unit in a sub-row: consecutive when W is odd, in the even /
                    // odd arrays when W is even (dd_kernel_gs.cu: Gs::DI)
                    const uint32_t base = off >> 5, pp = base & 1u, hh = base >> 1;
                    const uint32_t v0 = (W % 2) ? base : pp * (row_units / 2) + hh;
                    const uint32_t v1 = (W % 2) ? 0u : (1u - pp) * (row_units / 2) + hh + pp;
                    en[2 * i + 1] = (off & 31u) | (v0 << 8) | (v1 << 20);
                }
                row_idx += g.npat;
            }
            te[0].pad[5] = row_idx;   // rows in use in this stage
        }
    }
    p->var = Variant{5, DB, TB, 640, 32, 8, nbits, 0, 4, {cc, 0, 0, 0}, 1 << nbits, np, true, true, ubr, nsubr};
    p->pairs = false;
    p->gs = true;
    p->gs_G = G;
    p->gs_rows = rows;
    p->gs_row_units = row_units;
    p->gs_raw_sub = raw_sub;
    p->gs_nsr = nsr;
    p->gs_nsp = nsp;
    p->gs_patch = patch;
    p->long_mode = true;
    p->patch = patch;
    p->max_span_end = max_end;
    p->sub_slot = raw_sub;
    p->raw_slot = raw_sub * nsubr;
    p->lane_slot = p->raw_slot;
    p->cc = cc;
    p->nstages = nsr;
    p->ngroups = 1;
    p->group_cols = ents_pad;
    p->nblk = nblk;
    p->nchans_pad = ents_pad;
    p->smem_bytes = gs_smem_bytes(nbits, G, cc, rows, row_units, raw_sub, nsr, nsp, patch);
    p->span.swap(span);
    p->rel.swap(rel);
    p->gs_tab.swap(tab);
    p->live.swap(live);
    p->nlive = nlive;
    p->final32 = static_cast<int64_t>(nlive) * vmax > 65535;
    return DD_OK;
}

int64_t gr_smem_bytes(int nbits, int G, int nstages, int stage_bytes, bool patch)
{
    int64_t b = 128 + (patch ? 16 * static_cast<int64_t>(kBpPatchBytes) : 0);
    b += nstages * align_up((static_cast<int64_t>(gr_max_groups_per_stage(nbits, G)) * 16 + 16) * 8, 128);   // offset entries + trailer
    b += static_cast<int64_t>(nstages) * stage_bytes;                                                          // rows
    return b;
}

// Variant 6 -- group rows in device memory (dd_kernel_gr.cu).  Groups of G adjacent live channels; per group the
// distinct tuples (delta_1 .. delta_{G-1}), delta_i = delay[d][c_i] - delay[d][c_0], over the WHOLE DM list: one row
// R[t] = sum_i x[c_i][t + delta_i] per tuple is made by a pre-pass, every trial adds the row of its own tuple at the
// delay of c_0.  A stage holds, per DM block, the spans of the rows its 16 trials use, packed one after the other.
dd_status build_tiles_gr(dd_plan_s *p, int G)
{
    const int nrows = p->nchans, ndm = p->ndm, nbits = p->nbits;
    if (G == 0)
        G = 4;
    if (p->group_size > 0 || p->in_planes > 0 || (G != 2 && G != 4) || (nbits == 2 && G != 4))
        return DD_ERR_SMEM;
    std::vector<int32_t> live;
    for (int c = 0; c < nrows; ++c)
        if (p->keep.empty() || p->keep[c])
            live.push_back(c);
    const int nlive = static_cast<int>(live.size());
    if (nlive == 0)
        return DD_ERR_SMEM;
    const int W = nbits == 2 ? kGrW2 : 3, TB = 1024 * W, DB = 16;
    const int np = nbits == 2 ? 12 : (nbits == 4 ? 16 : 20);
    const int uw = gr_unit_words(nbits, G), ub = uw * 4;
    const int nfg = gr_flush_groups(nbits, G), gmax = gr_max_groups_per_stage(nbits, G), gq = gr_group_quantum(nbits, G);
    const int au = (ub % 16 == 0) ? 1 : 2;   // spans start and end on whole 16 bytes: pairs of units when a unit is 8 (mod 16) bytes
    const int64_t vmax = (1 << nbits) - 1;
    if (static_cast<int64_t>(nlive) * vmax >= (int64_t(1) << np))
        return DD_ERR_SMEM;
    const int ngr = (nlive + G - 1) / G;
    const int ents_pad = static_cast<int>(align_up(ngr, nfg));
    const int nblk = (ndm + DB - 1) / DB;

    // rows: every tuple of every group, in group order; per (trial, group) the row of the trial's tuple
    struct Tuple {
        int32_t d[4];
        bool operator<(const Tuple &o) const { return std::lexicographical_compare(d, d + 4, o.d, o.d + 4); }
        bool operator==(const Tuple &o) const { return std::equal(d, d + 4, o.d); }
    };
    std::vector<int32_t> prow;                                       // [n_rows][8] {c_0..c_3, delta_0..delta_3}
    std::vector<int32_t> row_of(static_cast<size_t>(ndm) * ngr);     // [d][q] global row index
    std::vector<Tuple> tup(ndm), uniq;
    for (int q = 0; q < ngr; ++q) {
        const int cnt = std::min(G, nlive - q * G);
        int32_t ch[4] = {-1, -1, -1, -1};
        for (int i = 0; i < cnt; ++i)
            ch[i] = live[q * G + i];
        for (int d = 0; d < ndm; ++d) {
            const int32_t *row = p->delay.data() + static_cast<size_t>(d) * nrows;
            Tuple t{{0, 0, 0, 0}};
            for (int i = 1; i < cnt; ++i) {
                t.d[i] = row[ch[i]] - row[ch[0]];
                if (t.d[i] < 0 || t.d[i] > (1 << 26))   // (never for a descending band; refused all the same)
                    return DD_ERR_SMEM;
            }
            tup[d] = t;
        }
        uniq = tup;
        std::sort(uniq.begin(), uniq.end());
        uniq.erase(std::unique(uniq.begin(), uniq.end()), uniq.end());
        const int32_t base = static_cast<int32_t>(prow.size() / 8);
        for (const Tuple &t : uniq) {
            prow.insert(prow.end(), ch, ch + 4);
            prow.insert(prow.end(), t.d, t.d + 4);
        }
        for (int d = 0; d < ndm; ++d)
            row_of[static_cast<size_t>(d) * ngr + q] =
                base + static_cast<int32_t>(std::lower_bound(uniq.begin(), uniq.end(), tup[d]) - uniq.begin());
        if (prow.size() / 8 > (size_t(1) << 28))
            return DD_ERR_SMEM;
    }
    const int64_t n_rows = static_cast<int64_t>(prow.size() / 8);
    {   // behind the rows: the first row of every group, and the row count (the builder works group by group)
        std::vector<int32_t> gbase;
        int32_t last = -1;
        for (int64_t r = 0; r < n_rows; ++r)
            if (r == 0 || prow[8 * r] != last) {   // c_0 changes from group to group
                gbase.push_back(static_cast<int32_t>(r));
                last = prow[8 * r];
            }
        gbase.push_back(static_cast<int32_t>(n_rows));
        prow.insert(prow.end(), gbase.begin(), gbase.end());
    }

    // per (DM block, group): the rows in use and the staged span of the group's first channel
    struct Use {
        int32_t start = 0, nbytes = 0, off[16];
        int nrow = 0;
        int32_t rows[16];
        uint8_t which[16];
    };
    auto analyse = [&](int b, int q, Use &u) -> bool {
        u = Use();
        if (q >= ngr) {   // padded group: the all-zero row, every window at its start
            u.nrow = 1;
            u.rows[0] = static_cast<int32_t>(n_rows);
            u.nbytes = static_cast<int32_t>(align_up(TB / 32 + 1, au)) * ub;
            for (int i = 0; i < DB; ++i)
                u.which[i] = 0, u.off[i] = 0;
            return true;
        }
        const int c0 = live[q * G];
        int32_t dmin = std::numeric_limits<int32_t>::max(), dmax = 0, d0s[16];
        for (int i = 0; i < DB; ++i) {
            const int d = std::min(b * DB + i, ndm - 1);   // the last block is padded with its last trial
            d0s[i] = p->delay[static_cast<size_t>(d) * nrows + c0];
            dmin = std::min(dmin, d0s[i]);
            dmax = std::max(dmax, d0s[i]);
            const int32_t r = row_of[static_cast<size_t>(d) * ngr + q];
            int f = -1;
            for (int k = 0; k < u.nrow && f < 0; ++k)
                if (u.rows[k] == r)
                    f = k;
            if (f < 0) {
                f = u.nrow++;
                u.rows[f] = r;
            }
            u.which[i] = static_cast<uint8_t>(f);
        }
        u.start = dmin / (32 * au) * (32 * au);
        if (dmax - u.start > (1 << 20))
            return false;
        const int64_t nunits = align_up(TB / 32 + (dmax - u.start) / 32 + 1, au);   // the funnel shift reads one unit further
        u.nbytes = static_cast<int32_t>(nunits * ub);
        for (int i = 0; i < DB; ++i)
            u.off[i] = d0s[i] - u.start;
        return true;
    };
    // pass 1: the largest group; then the byte budget of a stage: a ring of three (two if a single group needs more),
    // output patches for 2- and 4-bit input when the ring still holds the largest group beside them
    Use u;
    int64_t max_group = 0, max_end = 0;   // max_group: bytes of the largest quantum of gq consecutive groups
    int max_qrows = 0;
    for (int b = 0; b < nblk; ++b) {
        for (int q0 = 0; q0 < ents_pad; q0 += gq) {
            int64_t qb = 0;
            int qr = 0;
            for (int q = q0; q < q0 + gq; ++q) {
                if (!analyse(b, q, u))
                    return DD_ERR_SMEM;
                qb += static_cast<int64_t>(u.nrow) * u.nbytes;
                qr += u.nrow;
                max_end = std::max<int64_t>(max_end, static_cast<int64_t>(u.start) + u.nbytes / ub * 32);
            }
            max_group = std::max(max_group, qb);
            max_qrows = std::max(max_qrows, qr);
        }
    }
    if (max_qrows > 48)
        return DD_ERR_SMEM;
    int nst = 0;
    bool patch = false;
    int64_t stage_bytes = 0;
    // ring depth: two large stages beat three smaller ones except for the 9-plane rows of 8-bit pairs (measured with 2 / 3 /
    // 4 stages: cfg2 7.63 / 8.11 / 8.94 ms, cfg4 69.9 / 72.8 / 79.7, cfg5 143.9 / 146.0 / 151.9, cfg3 193 / 185 / 194)
    const int ns_pref = (nbits == 8 && G == 2) ? 3 : 2;
    const int cand[3][2] = {{ns_pref, 1}, {ns_pref, 0}, {2, 0}};
    for (const auto &cd : cand) {
        if (cd[1] && nbits == 8)
            continue;
        const int64_t fixed = gr_smem_bytes(nbits, G, cd[0], 0, cd[1] != 0);
        const int64_t budget = (kMaxDynSmem - fixed) / cd[0] / 128 * 128;
        if (budget >= max_group && budget > 0) {
            nst = cd[0], patch = cd[1] != 0, stage_bytes = std::min<int64_t>(budget, (1 << 20) - 128);
            break;
        }
    }
    if (nst == 0)
        return DD_ERR_SMEM;
    // pass 2: consecutive groups are packed into a stage until its bytes, 48 rows (3 per producer warp) or gmax groups
    // are reached; stage_of[b] lists the first group of every stage of block b
    std::vector<std::vector<int32_t>> first(nblk);
    int nstg_max = 0, rs = 1;
    for (int b = 0; b < nblk; ++b) {
        int64_t bytes = 0;
        int rows = 0, groups = 0;
        for (int q0 = 0; q0 < ents_pad; q0 += gq) {   // a quantum of gq groups at a time
            int64_t gb = 0;
            int gr_rows = 0;
            for (int q = q0; q < q0 + gq; ++q) {
                analyse(b, q, u);
                gb += static_cast<int64_t>(u.nrow) * u.nbytes;
                gr_rows += u.nrow;
            }
            if (q0 == 0 || groups + gq > gmax || rows + gr_rows > 48 || bytes + gb > stage_bytes) {
                first[b].push_back(q0);
                bytes = 0, rows = 0, groups = 0;
            }
            bytes += gb, rows += gr_rows, groups += gq;
            rs = std::max(rs, rows);
        }
        first[b].push_back(ents_pad);
        nstg_max = std::max(nstg_max, static_cast<int>(first[b].size()) - 1);
    }
    // pass 3: per block a header {stages, groups of the first stage} and the span list [nstg_max][rs]; offsets
    // [nblk][nstg_max][gmax * DB entries + a trailer whose first word is the group count of the NEXT stage]
    const size_t span_blk = static_cast<size_t>(nstg_max) * rs + 1, rel_stage = (static_cast<size_t>(gmax) * DB + DB) * 8;
    std::vector<SpanMeta> span(static_cast<size_t>(nblk) * span_blk, SpanMeta{0, 0, 0, 0});
    std::vector<uint8_t> rel(static_cast<size_t>(nblk) * nstg_max * rel_stage, 0);
    for (int b = 0; b < nblk; ++b) {
        const int nstg = static_cast<int>(first[b].size()) - 1;
        span[b * span_blk] = SpanMeta{nstg, first[b][1] - first[b][0], 0, 0};
        for (int k = 0; k < nstg; ++k) {
            SpanMeta *sl = span.data() + b * span_blk + 1 + static_cast<size_t>(k) * rs;
            uint32_t *en = reinterpret_cast<uint32_t *>(rel.data() + (static_cast<size_t>(b) * nstg_max + k) * rel_stage);
            en[2 * gmax * DB] = k + 1 < nstg ? static_cast<uint32_t>(first[b][k + 2] - first[b][k + 1]) : 0u;   // the trailer
            int slot = 0;
            int32_t dst = 0;
            for (int q = first[b][k]; q < first[b][k + 1]; ++q) {
                analyse(b, q, u);
                uint32_t *eg = en + static_cast<size_t>(q - first[b][k]) * DB * 2;
                for (int i = 0; i < DB; ++i) {
                    const uint32_t off = static_cast<uint32_t>(u.off[i]);
                    eg[2 * i] = static_cast<uint32_t>(dst + u.which[i] * u.nbytes) + (off >> 5) * static_cast<uint32_t>(ub);
                    eg[2 * i + 1] = off & 31u;
                }
                for (int j = 0; j < u.nrow; ++j) {
                    sl[slot++] = SpanMeta{u.start / 32 * ub, u.nbytes, u.rows[j], dst};
                    dst += u.nbytes;
                }
            }
        }
    }
    const int cc = gmax;
    p->var = Variant{6, DB, TB, 512, 32, 8, nbits, 0, 4, {cc, 0, 0, 0}, 1 << nbits, np, true, true, ub, 1};
    p->pairs = false;
    p->gs = false;
    p->gr = true;
    p->gs_G = G;
    p->long_mode = true;
    p->patch = patch;
    p->max_span_end = max_end;
    p->sub_slot = static_cast<int>(stage_bytes);
    p->raw_slot = static_cast<int>(stage_bytes);
    p->lane_slot = p->raw_slot;
    p->rows_per_chunk = rs;
    p->gr_stage_slots = nstg_max;
    p->cc = cc;
    p->nstages = nst;
    p->ngroups = 1;
    p->group_cols = ents_pad;
    p->nblk = nblk;
    p->nchans_pad = ents_pad;
    p->smem_bytes = gr_smem_bytes(nbits, G, nst, static_cast<int>(stage_bytes), patch);
    p->span.swap(span);
    p->rel.swap(rel);
    p->live.swap(live);
    p->nlive = nlive;
    p->prow.swap(prow);
    p->n_prows = n_rows;
    p->final32 = static_cast<int64_t>(nlive) * vmax > 65535;
    return DD_OK;
}

// Variant 5 with the group size and the groups per stage of dd_set_tuning, else the first compiled shape that fits.
static dd_status build_tiles_gs_auto(dd_plan_s *p)
{
    static const int shapes[3][2][2][2] = {
        /* 2-bit */ {{{2, 16}, {2, 16}}, {{4, 4}, {4, 4}}},
        /* 4-bit */ {{{2, 8}, {2, 8}}, {{4, 4}, {4, 4}}},
        /* 8-bit */ {{{2, 4}, {2, 2}}, {{4, 2}, {4, 1}}},
    };
    const int wi = p->nbits == 2 ? 0 : (p->nbits == 4 ? 1 : 2);
    for (int gi = 1; gi >= 0; --gi) {   // groups of four first
        for (int ci = 0; ci < 2; ++ci) {
            const int G = shapes[wi][gi][ci][0], cc = shapes[wi][gi][ci][1];
            if ((p->gs_force_G && p->gs_force_G != G) || (p->gs_force_cc && p->gs_force_cc != cc))
                continue;
            if (build_tiles_gs(p, G, cc) == DD_OK)
                return DD_OK;
        }
    }
    p->gs = false;
    return DD_ERR_SMEM;
}

dd_status build_tiles(dd_plan_s *p)
{
    p->pairs = false;
    p->gs = false;
    if (p->force_variant == 4)
        return build_tiles_pairs(p);
    if (p->force_variant == 5)
        return build_tiles_gs_auto(p);
    p->gr = false;
    if (p->force_variant == 6)
        return build_tiles_gr(p, p->gs_force_G);
    // Default for 4- and 8-bit input: pair rows (variant 4, 15-17 % faster on cfg3-5), unless the plan sums channel
    // groups (sub-band steps), the caller promised small samples (dd_set_input_max: variant 3 then skips planes), or
    // the pair planner cannot serve the table (then variant 3 and the others are tried as before).  2-bit input
    // stays on variant 3: the pair rows gain nothing there.
    if (p->force_variant == 0 && p->group_size == 0 && p->in_planes == 0 && p->nchans >= 128) {
        // Default: group rows (variant 6) when their cost model says so -- rows of four channels first, pairs if those do
        // not fit shared memory (large delay spreads) -- else, for 4- and 8-bit input, the pair rows of variant 4.
        for (int G : {4, 2}) {
            if (p->gs_force_G && p->gs_force_G != G)
                continue;
            if (build_tiles_gr(p, G) != DD_OK)
                continue;
            // cost per 32 output samples, in ALU lane-operations: the bit-plane kernel adds nbits plane words per trial
            // and channel (a shift + 2.13 LOP3 each); with group rows every trial adds pin words per group, every row
            // costs its G shifted loads and ripple adders plus its bytes written (3.4 lane-operations per byte: 5.5 TB/s
            // against 18.6e12 lane-operations/s; reading them back overlaps with the adds).  Calibrated on a B200: model
            // 0.57 / 0.55 / 0.69 / 0.87 of the bit-plane kernel for cfg5 / cfg4 / cfg3 (pairs) / cfg2, measured 0.64 / 0.62 /
            // 0.75 / 0.87.
            const double pin = p->nbits + (G == 2 ? 1 : 2), ngr = (p->nlive + G - 1) / G;
            const double direct = 3.13 * p->ndm * static_cast<double>(p->nlive) * p->nbits;
            const double rows = static_cast<double>(p->n_prows) * (G * p->nbits + 2.0 * (G - 1) * (p->nbits + 1) +
                                                                  3.4 * 4.0 * gr_unit_words(p->nbits, G));
            const double grouped = 3.13 * p->ndm * ngr * pin + rows;
            // ... and the rows must not swamp the memory system: written once, read about 1.5 times at ~4 TB/s (11.6
            // lane-operations per byte of row); cfg3 with rows of four (393 GB of rows, each used by 4 trials only)
            // measured 590 ms against 185 ms with pairs
            const double row_bytes = static_cast<double>(p->n_prows) * 4.0 * gr_unit_words(p->nbits, G);
            if (grouped < 0.9 * direct && 11.6 * row_bytes < 0.9 * direct)
                return DD_OK;
            p->gr = false;
        }
        p->gr = false;
        if ((p->nbits == 4 || p->nbits == 8) && p->gs_force_G == 0 && build_tiles_pairs(p) == DD_OK)
            return DD_OK;
    }
    p->pairs = false;
    const int nrows = p->nchans, ndm = p->ndm, nbits = p->nbits;
    // the channels that are summed (PAPER.md:113 kill mask): the kernels iterate over this list only
    std::vector<int32_t> live;
    for (int c = 0; c < nrows; ++c)
        if (p->keep.empty() || p->keep[c])
            live.push_back(c);
    const int nchans = static_cast<int>(live.size());
    // channel groups (sub-bands): position range [gbeg[g], gbeg[g+1]) of the live list
    const int gsize = p->group_size > 0 ? p->group_size : std::max(nrows, 1);
    const int ngroups = (nrows + gsize - 1) / gsize;
    std::vector<int> gbeg(ngroups + 1, 0);
    for (int c : live)
        ++gbeg[c / gsize + 1];
    int gmax = 0;
    for (int g = 0; g < ngroups; ++g) {
        gmax = std::max(gmax, gbeg[g + 1]);
        gbeg[g + 1] += gbeg[g];
    }
    const int64_t vmax = (1 << nbits) - 1;
    const int64_t top = static_cast<int64_t>(gmax) * vmax;   // largest possible sum
    p->final32 = top > 65535;

    for (const Variant &v : kVariants) {
        // samples per 16 staged bytes (the bulk-copy granularity): of the packed row, or of a bit-plane sub-row
        const int A = v.bitplane ? (16 / v.unit_bytes) * 32 : 128 / nbits;
        if (!(v.nbits_mask & (1 << nbits)) || (v.max_sum_bits < 32 && top >= (int64_t(1) << v.max_sum_bits)))
            continue;
        if (p->force_variant && v.id != p->force_variant)
            continue;
        if (ngroups > 1 && !v.bitplane)
            continue;   // channel groups are served by the bit-plane kernel only
        p->var = v;
        // Bit planes: with many channels per group the LONG instantiation flushes the pending words only every
        // kBpFlushStages stages (channel list padded to whole flush groups) and, for 8-bit input -- four times the
        // work of 2-bit input per channel, the epilogue a per-mille effect -- spends the shared memory of the
        // output patches on a deeper ring.  With few channels (sub-band steps) the epilogue dominates.
        const int fl = v.bitplane ? kBpFlushStages(nbits) : 1;
        p->long_mode = v.bitplane && gmax >= 8 * v.cc[0] * fl;
        p->patch = v.bitplane && (!p->long_mode || nbits < 8);
        const int DB = v.DB;
        const int nblk = (ndm + DB - 1) / DB;
        const int64_t rel_limit = v.rel_bytes == 2 ? 65535 : (int64_t(1) << 26);
        // pass 1: the staged span of every (DM block, channel): [dmin rounded down to the copy granularity,
        // dmax + time block + over-fetch)
        std::vector<SpanMeta> span0(static_cast<size_t>(nblk) * nchans);
        int64_t max_bytes = 0, max_end = 0;
        bool ok = true;
        for (int b = 0; b < nblk && ok; ++b) {
            for (int c = 0; c < nchans; ++c) {
                int32_t dmin = std::numeric_limits<int32_t>::max(), dmax = 0;
                for (int i = 0; i < DB; ++i) {
                    const int d = std::min(b * DB + i, ndm - 1);   // pad the last block with its last DM
                    const int32_t dl = p->delay[static_cast<size_t>(d) * nrows + live[c]];
                    dmin = std::min(dmin, dl);
                    dmax = std::max(dmax, dl);
                }
                const int32_t start = dmin / A * A;
                const int64_t need = static_cast<int64_t>(v.TB) + (dmax - start) + v.tail;
                const int64_t nbytes = v.bitplane ? align_up(need, A) / 32 * v.unit_bytes   // per sub-row
                                                  : align_up(need, A) * nbits / 8;
                if (dmax - start > rel_limit || nbytes > (1 << 19)) {
                    ok = false;
                    break;
                }
                SpanMeta &m = span0[static_cast<size_t>(b) * nchans + c];
                m.start = start;
                m.nbytes = static_cast<int32_t>(nbytes);
                m.row = live[c];
                m.pad = 0;
                max_bytes = std::max(max_bytes, nbytes);
                max_end = std::max(max_end, start + (v.bitplane ? nbytes / v.unit_bytes * 32 : nbytes * 8 / nbits));
            }
        }
        if (!ok)
            continue;
        p->max_span_end = max_end;
        p->sub_slot = static_cast<int>(max_bytes);
        p->raw_slot = static_cast<int>(max_bytes) * v.nsub;
        p->lane_slot = static_cast<int>(max_bytes * v.lane_bits / nbits);
        int cc = 0;
        for (p->nstages = v.raw_stages; p->nstages >= 2 && cc == 0; --p->nstages) {   // deepest ring that fits
            for (int k = 0; k < 4 && v.cc[k] > 0; ++k) {
                const int cand = v.cc[k];
                if (!v.pad_chunks && k + 1 < 4 && v.cc[k + 1] > 0 && v.cc[k + 1] >= nchans)
                    continue;   // a smaller stage already covers every channel
                const int64_t tx = static_cast<int64_t>(cand) * p->raw_slot + static_cast<int64_t>(cand) * DB * v.rel_bytes;
                if (smem_layout_bytes(p, cand) <= kMaxDynSmem && tx < (1 << 20)) {
                    cc = cand;
                    break;
                }
            }
            if (cc)
                break;
        }
        if (cc < 1)
            continue;
        // pass 2: per (DM, column) the position of that DM's window inside the staged span.  Column k of group g
        // is the k-th live channel of the group; columns past the group's live count are padded (zero) channels.
        const int group_cols = v.pad_chunks ? static_cast<int>(align_up(gmax, cc * (p->long_mode ? fl : 1))) : gmax;
        const int nchans_pad = ngroups * group_cols;
        std::vector<SpanMeta> span(static_cast<size_t>(nblk) * nchans_pad);
        std::vector<uint8_t> rel(static_cast<size_t>(nblk) * nchans_pad * DB * v.rel_bytes);
        for (int b = 0; b < nblk; ++b) {
            for (int col = 0; col < nchans_pad; ++col) {
                SpanMeta &m = span[static_cast<size_t>(b) * nchans_pad + col];
                const size_t base = (static_cast<size_t>(b) * nchans_pad + col) * DB;
                const int g = col / std::max(group_cols, 1), k = col - g * group_cols;
                const uint32_t slot_off = static_cast<uint32_t>(k % cc) * static_cast<uint32_t>(p->raw_slot);
                if (k >= gbeg[g + 1] - gbeg[g]) {   // padded channel: a whole slot of zeros, every window at its start
                    m.start = 0;
                    m.pad = 0;
                    if (v.bitplane) {   // staged from the all-zero row the launcher keeps behind the input rows
                        m.row = nrows;
                        m.nbytes = p->sub_slot;
                    } else {
                        m.row = 0;
                        m.nbytes = -p->raw_slot;   // negative: stage from the zero buffer
                    }
                    for (int i = 0; i < DB; ++i) {
                        uint32_t *e = reinterpret_cast<uint32_t *>(rel.data()) + (base + i) * 2;
                        e[0] = slot_off;
                        e[1] = 0;
                    }
                    continue;
                }
                const int c = gbeg[g] + k;   // position in the live list
                m = span0[static_cast<size_t>(b) * nchans + c];
                const int32_t start = m.start;
                if (v.bitplane) {   // the kernel wants the byte offset of the span inside a bit-plane sub-row (tile 0)
                    m.pad = start;
                    m.start = start / 32 * v.unit_bytes;
                }
                for (int i = 0; i < DB; ++i) {
                    const int d = std::min(b * DB + i, ndm - 1);
                    const uint32_t off = static_cast<uint32_t>(p->delay[static_cast<size_t>(d) * nrows + live[c]] - start);
                    if (v.rel_bytes == 2) {
                        reinterpret_cast<uint16_t *>(rel.data())[base + i] = static_cast<uint16_t>(off);
                    } else if (v.rel_bytes == 4) {
                        reinterpret_cast<uint32_t *>(rel.data())[base + i] = off * 4u;
                    } else {   // bit planes: 32 samples per unit of unit_bytes
                        uint32_t *e = reinterpret_cast<uint32_t *>(rel.data()) + (base + i) * 2;
                        e[0] = slot_off + (off >> 5) * static_cast<uint32_t>(v.unit_bytes);
                        e[1] = off & 31u;
                    }
                }
            }
        }
        p->cc = cc;
        p->ngroups = ngroups;
        p->group_cols = group_cols;
        p->nblk = nblk;
        p->nchans_pad = nchans_pad;
        p->smem_bytes = smem_layout_bytes(p, cc);
        p->span.swap(span);
        p->rel.swap(rel);
        p->live.swap(live);
        p->nlive = nchans;
        return DD_OK;
    }
    return DD_ERR_SMEM;
}

}  // namespace dd
