// host_plan.h -- host-side construction of the kernel plans (tile schedule, schedule-ordered coefficient
// tables, reaction chunks and incidence lists) appended to the single device block of a mechanism.
// Private to libcrf.so.
#pragma once
#include <algorithm>
#include <cstring>
#include <vector>

#include "../../include/crf_diag.h"
#include "crf_internal.h"

struct BlockBuilder {
    std::vector<unsigned char> bytes;
    template <class T>
    size_t add(const std::vector<T> &v)
    {
        size_t off = (bytes.size() + 255) & ~size_t(255);
        bytes.resize(off + std::max<size_t>(v.size(), 1) * sizeof(T));
        if (!v.empty()) std::memcpy(bytes.data() + off, v.data(), v.size() * sizeof(T));
        return off;
    }
};

// Offsets (into the block) of what a plan points to; resolved to device pointers after the upload.
struct TransportPlanOffsets {
    int W = 0, PPL = 0, NsP = 0, nb = 0, n_wilke = 0, n_rounds = 0, stage_bytes = 0;
    int TS = 8, nbp = 0;  // tile edge and species blocks of the pair phase
    int small_n = 0;
    size_t small = 0, rounds = 0, pair_coef = 0, wilke_cP = 0, sp = 0, Ddiag = 0;
};
struct RatesPlanOffsets {
    int W = 0, Rc = 0, n_chunks = 0;
    size_t chunk = 0, rc = 0, rs = 0, inc_ptr = 0, inc = 0, troe = 0, gco = 0, hco = 0;
};

struct RatesSmemPlanOffsets {
    int W = 0, PPL = 0, maxown = 0, Rc = 0, n_chunks = 0, stage_bytes = 0;
    size_t chunk = 0, stage = 0, gco = 0, hco = 0;
};

// `opt` is the explicit plan request of crf_mech_create_ex (all zero = automatic); a builder that cannot honour
// the request returns an empty plan (W = 0) and crf_mech_create_ex reports CRF_EUNSUPPORTED.
struct RatesGroupPlanOffsets {
    int W = 0, PPL = 0, maxown = 0, Rc = 0, q_rows = 0, tm_cols = 0, n_chunks = 0, stage_bytes = 0;
    double log2_c0 = 0.0;
    size_t chunk = 0, stage = 0, gco = 0, hco = 0, own = 0;
};

TransportPlanOffsets build_transport_plan(const crf_tables *t, const crf_plan_options &opt, BlockBuilder &b);
RatesPlanOffsets build_rates_plan(const crf_tables *t, const crf_plan_options &opt, BlockBuilder &b);
RatesSmemPlanOffsets build_rates_smem_plan(const crf_tables *t, const crf_plan_options &opt, BlockBuilder &b);
RatesGroupPlanOffsets build_rates_group_plan(const crf_tables *t, const crf_plan_options &opt, BlockBuilder &b);
