// K_score instantiations for L = 4 pressure levels (see dyplan_score.cuh).
#define DYPLAN_SCORE_L 4
#include "dyplan_score.cuh"
