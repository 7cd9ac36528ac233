// K_fscore for a padded level count of 4 (see dyplan_fscore.cuh)
#define DYPLAN_FSCORE_L 4
#include "dyplan_fscore.cuh"
