// K_score instantiations for L = 2 pressure levels (see dyplan_score.cuh).
#define DYPLAN_SCORE_L 2
#include "dyplan_score.cuh"
