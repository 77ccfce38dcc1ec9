// sg_tmpl_shard.cu — one shard of the precompiled template instances: compiled SG_NSHARDS times with -DSG_SHARD=k
// (paper_1410_6685_b200/build.py).  Shard k instantiates the kernels of the instances whose index i satisfies
// i % SG_NSHARDS == k; sg_kernels.cu merges the shards' tables into the registry.
#include "sg_tmpl_launch.cuh"

#ifndef SG_SHARD
#error "compile with -DSG_SHARD=<0..SG_NSHARDS-1>"
#endif
#ifndef SG_TEMPLATES_INC
#define SG_TEMPLATES_INC "sg_templates_gen.inc"      // tuning experiments compile a shard against another instance list
#endif

namespace {

using namespace sgk;

// Each SG_TEMPLATE(index, name, unroll, min_blocks, row_unroll, stages, {program}) in the generated file defines a policy type.
// The program initialisers are written by paper_1410_6685_b200/gen_templates.py from the plan builder's own canonical
// output, so a registered chain always matches its signature.
#define SG_TEMPLATE(IDX, NAME, UNROLL, MINB, ROWU, STAGES, ...)                      \
    struct T_##NAME {                                                                \
        static constexpr SgProg prog = __VA_ARGS__;                                  \
        static constexpr int unroll = UNROLL, min_blocks = MINB, row_unroll = ROWU, stages = STAGES;  \
    };
#include SG_TEMPLATES_INC
#undef SG_TEMPLATE

#define SG_TEMPLATE(IDX, NAME, UNROLL, MINB, ROWU, STAGES, ...) EntryOf<T_##NAME, (IDX) % SG_NSHARDS == SG_SHARD>::make(#NAME),
const Entry g_shard_entries[] = {
#include SG_TEMPLATES_INC
};
#undef SG_TEMPLATE

}  // namespace

#define SG_CAT2(a, b) a##b
#define SG_CAT(a, b) SG_CAT2(a, b)
const sgk::Entry* SG_CAT(sgk_shard_entries_, SG_SHARD)(int* n) {
    *n = (int)(sizeof(g_shard_entries) / sizeof(g_shard_entries[0]));
    return g_shard_entries;
}
