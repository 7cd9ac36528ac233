// K_score instantiations for L = 5 pressure levels (see dyplan_score.cuh).
#define DYPLAN_SCORE_L 5
#include "dyplan_score.cuh"
