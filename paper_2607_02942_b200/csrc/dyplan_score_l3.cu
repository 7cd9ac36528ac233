// K_score instantiations for L = 3 pressure levels (see dyplan_score.cuh).
#define DYPLAN_SCORE_L 3
#include "dyplan_score.cuh"
