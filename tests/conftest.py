"""pytest configuration: the `gpu` marker and shared helpers.

`-m "not gpu"` : oracle vs its pins, host logic, C-ABI symbol check, gloo world_size-2 sharding.
`-m gpu`       : parity of the CUDA path (through the C ABI) with the CPU oracle on a B200.
"""
import sys
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

GOLDEN = Path(__file__).resolve().parent / "golden"


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); parity tests proper")


# direction of travel source -> target, d = 0..7 = N, NE, E, SE, S, SW, W, NW (C-2);
# restated here (not imported) so that tests do not inherit an indexing mistake from either side
OFFSETS = [(0, -1), (1, -1), (1, 0), (1, 1), (0, 1), (-1, 1), (-1, 0), (-1, -1)]


def unpack_bitmap(words: np.ndarray, W: int) -> np.ndarray:
    """u32[H][ceil(W/32)] canonical bitmap -> bool[H][W] (bit x&31 of word x>>5, LSB = lowest x)."""
    words = np.ascontiguousarray(words, dtype="<u4")
    bits = np.unpackbits(words.view(np.uint8), axis=-1, bitorder="little")
    return bits[..., :W].astype(bool)


def pack_bitmap(mask: np.ndarray) -> np.ndarray:
    H, W = mask.shape
    Ww = (W + 31) // 32
    padded = np.zeros((H, Ww * 32), np.uint8)
    padded[:, :W] = mask
    return np.packbits(padded, axis=-1, bitorder="little").view("<u4").reshape(H, Ww).astype(np.uint32)


@pytest.fixture(scope="session")
def orc():
    from oracle import fire_oracle
    fire_oracle.build()
    return fire_oracle
