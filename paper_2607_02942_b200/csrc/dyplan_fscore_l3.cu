// K_fscore for a padded level count of 3 (see dyplan_fscore.cuh)
#define DYPLAN_FSCORE_L 3
#include "dyplan_fscore.cuh"
