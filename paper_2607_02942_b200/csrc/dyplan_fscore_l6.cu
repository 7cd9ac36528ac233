// K_fscore for a padded level count of 6 (see dyplan_fscore.cuh)
#define DYPLAN_FSCORE_L 6
#include "dyplan_fscore.cuh"
