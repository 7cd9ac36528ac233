// K_score instantiations for L = 6 pressure levels (see dyplan_score.cuh).
#define DYPLAN_SCORE_L 6
#include "dyplan_score.cuh"
