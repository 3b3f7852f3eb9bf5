"""bs_oracle_queue.py — TEST INFRASTRUCTURE ONLY.  The plain sequential definition of the SAVE / LOAD QUEUE
(SURVEY.md §8(f) NEXT-3).

What it follows.  PAPER.md §III.B.4:
  L136-138  "organizing asynchronous load and save into a kind of queuing system together with checkpoints to make
            sure that required data of a given computational task are already available in the memory, could
            maximize performance rate regarding IO operations."
  L132      a save is started after the data it saves is complete; L134 a load restores "the block sparse matrix and
            tensor structures" of what was saved.
The paper states no interface; the one below is this project's.  However the operations overlap
in time on the GPU, what a user may observe is fixed by PROGRAM ORDER, and that is what this model is — a dictionary:

  save(key, set, data)  the scratch store holds, under `key`, the wire-format-v1 stream of the set as it is at the
                        moment of the call (oracle.serialize); a later save under the same key replaces it
  save_layered(key, ..) the same for a layered set: the store holds its wire-format-v2 stream (oracle.v2.serialize)
  adopt(key, stream)    the store holds `stream` (bytes that came from elsewhere, either format) under `key`
  load(key)             the object identical to the one saved last under `key` (oracle.deserialize of the stored
                        stream); an unknown key is an error (ERR_ARG); a corrupt stream is ERR_CORRUPT
  load_layered(key)     the same for a key that holds a v2 stream; a key holds a stream of ONE format, asking for the
                        other is ERR_ARG
  forget(key)           the store drops `key`
  spill(key, path)      the file `path` holds exactly the bytes of the stream stored under `key` (saving =
                        serialization, then "writing the serialized data to a storage media"); the key stays in the store
  fill(key, path)       the store holds the bytes of the file under `key` (as adopt); a missing file is ERR_IO (-6)
  accounting            host_bytes_live = sum of the stored streams' lengths; host_bytes_peak = its maximum over the
                        calls so far; saves / loads = number of accepted calls; bytes_saved / bytes_loaded = stream
                        bytes moved by them

Nothing here is asynchronous, on purpose: the checkpoints of L138 exist to make the asynchronous execution
indistinguishable from this one.  Pins (tests/test_oracle_queue.py): a hand-traced sequence over the golden stream P7
(values typed in the test), the accounting against sums typed by hand, errors.  Unpinned: nothing.
Shares no code with the CUDA path; uses only oracle.serialize / oracle.deserialize (pinned in their own tests).
"""
from __future__ import annotations

import numpy as np

from . import bs_oracle as _v1
from . import bs_oracle_v2 as _v2


class QueueModel:
    def __init__(self):
        self.store: dict[int, np.ndarray] = {}
        self.saves = self.loads = 0
        self.bytes_saved = self.bytes_loaded = 0
        self.host_bytes_peak = 0
        self.bytes_spilled = self.bytes_filled = 0

    @property
    def host_bytes_live(self) -> int:
        return int(sum(len(s) for s in self.store.values()))

    def _account(self):
        self.host_bytes_peak = max(self.host_bytes_peak, self.host_bytes_live)

    def save(self, key: int, tensors, qn, dim, addr) -> np.ndarray:
        """addr = host addresses of the blocks (read NOW).  Returns the stored stream."""
        s = _v1.serialize(tensors, qn, dim, addr)
        self.store[int(key)] = s.copy()
        self.saves += 1
        self.bytes_saved += len(s)
        self._account()
        return self.store[int(key)]

    def save_layered(self, key: int, structs, layers, qn, dim, addr) -> np.ndarray:
        s = _v2.serialize(structs, layers, qn, dim, addr)
        self.store[int(key)] = s.copy()
        self.saves += 1
        self.bytes_saved += len(s)
        self._account()
        return self.store[int(key)]

    def adopt(self, key: int, stream) -> None:
        self.store[int(key)] = np.ascontiguousarray(stream, dtype=np.uint8).copy()
        self._account()

    @staticmethod
    def _is_v2(s) -> bool:
        return len(s) >= 12 and int(np.frombuffer(bytes(s[8:12]), "<u4")[0]) == 2     # the header's version word

    def _load(self, key: int, layered: bool) -> dict:
        if int(key) not in self.store:
            raise _v1.OracleError(_v1.ERR_ARG, "queue load: unknown key")
        s = self.store[int(key)]
        if self._is_v2(s) != layered:
            raise _v1.OracleError(_v1.ERR_ARG, "queue load: the key holds a stream of the other wire format")
        out = _v2.deserialize(s) if layered else _v1.deserialize(s)     # raises ERR_CORRUPT for a bad stream
        self.loads += 1
        self.bytes_loaded += len(s)
        return out

    def load(self, key: int) -> dict:
        return self._load(key, False)

    def load_layered(self, key: int) -> dict:
        return self._load(key, True)

    def forget(self, key: int) -> None:
        if int(key) not in self.store:
            raise _v1.OracleError(_v1.ERR_ARG, "queue forget: unknown key")
        del self.store[int(key)]

    def spill(self, key: int, path: str) -> int:
        if int(key) not in self.store:
            raise _v1.OracleError(_v1.ERR_ARG, "queue spill: unknown key")
        with open(path, "wb") as f:
            f.write(self.store[int(key)].tobytes())
        self.bytes_spilled += len(self.store[int(key)])
        return len(self.store[int(key)])

    def fill(self, key: int, path: str) -> int:
        try:
            with open(path, "rb") as f:
                raw = f.read()
        except OSError:
            raise _v1.OracleError(-6, "queue fill: cannot read the file")
        self.adopt(key, np.frombuffer(raw, np.uint8))
        self.bytes_filled += len(raw)
        return len(raw)

    def stats(self) -> dict:
        return dict(saves=self.saves, loads=self.loads, bytes_saved=self.bytes_saved, bytes_loaded=self.bytes_loaded,
                    host_bytes_live=self.host_bytes_live, host_bytes_peak=self.host_bytes_peak, keys_live=len(self.store))
