// K_score instantiations for L = 8 pressure levels (see dyplan_score.cuh).
#define DYPLAN_SCORE_L 8
#include "dyplan_score.cuh"
