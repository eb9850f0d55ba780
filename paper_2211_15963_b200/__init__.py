"""B200-native single-GPU step loop of the Digital Brain spiking-network simulator (arXiv 2211.15963).

The product is the CUDA library `libdb_b200.so` (C ABI in include/db_b200.h);
this package is its thin ctypes binding.  There is no CPU path.
"""
from .binding import (EXEC_AUTO, EXEC_KERNELS, EXEC_KERNELS_DEFERRED, EXEC_PERSISTENT, FIELD_G_AMPA, FIELD_G_GABAA, FIELD_G_GABAB,
                      FIELD_G_NMDA, FIELD_IEXT, FIELD_IOU, FIELD_OUTDEG, FIELD_REF, FIELD_RING, FIELD_TYPE, FIELD_V, DbError, Sim, load, lib_path)
from .build import build

__all__ = ["Sim", "DbError", "load", "build", "lib_path", "EXEC_AUTO", "EXEC_KERNELS", "EXEC_PERSISTENT", "EXEC_KERNELS_DEFERRED",
           "FIELD_V", "FIELD_G_AMPA", "FIELD_G_NMDA", "FIELD_G_GABAA", "FIELD_G_GABAB", "FIELD_REF", "FIELD_TYPE",
           "FIELD_RING", "FIELD_OUTDEG", "FIELD_IOU", "FIELD_IEXT"]
