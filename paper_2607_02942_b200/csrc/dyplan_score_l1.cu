// K_score instantiations for L = 1 pressure levels (see dyplan_score.cuh).
#define DYPLAN_SCORE_L 1
#include "dyplan_score.cuh"
