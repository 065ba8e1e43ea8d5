"""B200-native ODB hot path (group -> align -> collate), arxiv/paper_2606_19989.

The product is ``libodb.so`` (hand-written sm_100a CUDA behind the C ABI of ``include/odb.h``); this
package is its thin ctypes binding.  No CPU fallback exists: see ``binding.load``.
"""
from .binding import *  # noqa: F401,F403
from .binding import (  # noqa: F401
    Odb, OdbError, OdbLibraryError, OutputBuffers, SYMBOLS, library_path, load, make_params,
    odb_outputs, odb_params, odb_plan_info, status_string,
)
from .batches import StepBatches, StepStream  # noqa: F401,E402
from .stream import WorkerPool, plan_online  # noqa: F401,E402
