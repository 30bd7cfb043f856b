#define QM_TU_MODE 3
#include "qm_plane_tu.h"
