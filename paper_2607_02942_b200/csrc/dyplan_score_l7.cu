// K_score instantiations for L = 7 pressure levels (see dyplan_score.cuh).
#define DYPLAN_SCORE_L 7
#include "dyplan_score.cuh"
