// K_fscore for a padded level count of 8 (see dyplan_fscore.cuh)
#define DYPLAN_FSCORE_L 8
#include "dyplan_fscore.cuh"
