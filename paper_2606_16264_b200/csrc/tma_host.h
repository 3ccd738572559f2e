#pragma once
#include <cuda.h>

namespace tropical {
bool encode_pool_map(CUtensorMap* map, const void* base, long long rows, int D, int box_rows = 16);
bool encode_q_map(CUtensorMap* map, const void* base, int T, int Hq, int D, int box_heads, int box_tokens);
}  // namespace tropical
