// K_fscore for a padded level count of 2 (see dyplan_fscore.cuh)
#define DYPLAN_FSCORE_L 2
#include "dyplan_fscore.cuh"
