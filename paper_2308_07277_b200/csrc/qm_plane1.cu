#define QM_TU_MODE 1
#include "qm_plane_tu.h"
