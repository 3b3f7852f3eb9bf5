"""CPU oracle — TEST INFRASTRUCTURE ONLY (see bs_oracle.c header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this
package.  It imports nothing from paper_2412_04676_b200.
"""
from . import bs_oracle_dtype as dt  # noqa: F401  (element types other than fp64)
from . import bs_oracle_pkg as pkg  # noqa: F401  (self-contained packages)
from . import bs_oracle_v2 as v2  # noqa: F401  (wire format v2: structure-shared layers)
from . import bs_oracle_v3 as v3  # noqa: F401  (wire format v3: tensors of rank up to 4)
from .bs_oracle_queue import QueueModel  # noqa: F401  (save / load queue: the sequential definition)
from .bs_oracle import (  # noqa: F401
    ERR_ARG,
    ERR_CAPACITY,
    ERR_CORRUPT,
    ERR_UNSUPPORTED,
    OK,
    OracleError,
    deserialize,
    emit_header,
    emit_payload_range,
    header_bytes,
    plan,
    pool_bytes,
    serialize,
    serialized_size,
    stream_info,
    validate_set,
    validate_stream,
)
from .bs_oracle import build as _build_v1


def build(force: bool = False) -> str:
    """Compile every C file of the oracle (v1, v2 and package libraries)."""
    so = _build_v1(force)
    v2.build(force)
    v3.build(force)
    pkg.build(force)
    return so
