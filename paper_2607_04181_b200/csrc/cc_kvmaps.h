// cc_kvmaps.h -- TMA descriptors of the KV pools, one pair per replica (kernel parameters of the attention kernels).
// A replica may own its KV partition as a separate allocation (cc_layer_set_kv_partition); the
// rows of its requests then read their pages through ITS descriptor.  Without partitions all four are the same.
#pragma once
#include "cc_kernels.h"
#include <cuda.h>

struct CcKvMaps {
    CUtensorMap k[CC_MAXR];
    CUtensorMap v[CC_MAXR];
};
// box_rows: rows of one TMA box (one page of all kv heads: Hkv * 16; one page of one head: 16)
cudaError_t cc_make_kv_tensor_map(CUtensorMap* out, const void* pool, int n_pages, int Hkv, int Dh, int box_rows);
cudaError_t cc_make_kv_maps(CcKvMaps* out, const CcKv& kv, int Hkv, int Dh, int box_rows);
