// K_fscore for a padded level count of 1 (see dyplan_fscore.cuh)
#define DYPLAN_FSCORE_L 1
#include "dyplan_fscore.cuh"
