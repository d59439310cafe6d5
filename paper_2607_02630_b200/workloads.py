"""Seeded synthetic workloads shaped like the paper's offloads.

This module holds NO cipher arithmetic: it only draws bytes, keys, initial
counter blocks and lengths.  It serves both the oracle-side tests and the CUDA
path (tests, bench.py, smoke) so that the two are compared on identical inputs
while sharing no method code.  It imports neither ``oracle`` nor the CUDA
binding.

Shapes follow BASELINE.json ``configs`` and SURVEY.md section 8(d): payloads are
opaque request bodies (the paper's load generators ``redis-benchmark``/``ab``
send opaque payloads), block sizes are the paper's powers of two
from 4 KiB to 8 MiB (Table 2 at PAPER.md:356-369), concurrency is
tens of clients (50 at PAPER.md:350, 64 at PAPER.md:172).  Bytes are uniform
random because AES run time is data independent.

Generator: numpy Philox (counter based), key = (SEED_BASE + config index,
stream id), so any single request can be regenerated without the others.
"""
from __future__ import annotations

import dataclasses

import numpy as np

SEED_BASE = 260702630  # + config index (1..5), SURVEY.md section 8(d)

KIB = 1024
MIB = 1024 * 1024

# stream ids inside one config
_STREAM_KEYS = 1
_STREAM_ICBS = 2
_STREAM_LENS = 3
_STREAM_PAYLOAD0 = 1 << 20  # payload of request i uses stream _STREAM_PAYLOAD0 + i


def _rng(config_index: int, stream: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[SEED_BASE + config_index, stream]))


@dataclasses.dataclass
class Workload:
    """A batch of independent AES-CTR requests.

    keys[k]          : bytes, 16 or 32 long
    key_id[i]        : index into ``keys`` for request i
    icb[i]           : 16 bytes, the initial counter block of request i
    length[i]        : payload bytes of request i
    in_flight        : closed-loop window the config prescribes
    """

    name: str
    config_index: int
    keys: list
    key_id: np.ndarray
    icb: np.ndarray  # [n, 16] uint8
    length: np.ndarray  # [n] int64
    in_flight: int

    @property
    def n(self) -> int:
        return int(self.length.shape[0])

    @property
    def total_bytes(self) -> int:
        return int(self.length.sum())

    def key_of(self, i: int) -> bytes:
        return self.keys[int(self.key_id[i])]

    def icb_of(self, i: int) -> bytes:
        return self.icb[i].tobytes()

    def payload(self, i: int) -> np.ndarray:
        """Uniform random payload of request i (uint8, length[i])."""
        n = int(self.length[i])
        return payload_bytes(self.config_index, i, n)


def payload_bytes(config_index: int, request_index: int, n: int) -> np.ndarray:
    rng = _rng(config_index, _STREAM_PAYLOAD0 + request_index)
    return np.frombuffer(rng.bytes(n), dtype=np.uint8)


def _icbs_nonce_counter0(config_index: int, n: int) -> np.ndarray:
    """8 random nonce bytes || 8-byte big-endian counter starting at 0 (config 1)."""
    rng = _rng(config_index, _STREAM_ICBS)
    icb = np.zeros((n, 16), dtype=np.uint8)
    icb[:, :8] = rng.integers(0, 256, size=(n, 8), dtype=np.uint8)
    return icb


def _keys(config_index: int, sizes: list) -> list:
    rng = _rng(config_index, _STREAM_KEYS)
    return [rng.integers(0, 256, size=s, dtype=np.uint8).tobytes() for s in sizes]


def config1() -> Workload:
    """AES-128-CTR, one 64 KiB payload, one in flight (BASELINE.json configs[0])."""
    return Workload("c1_aes128_64KiB_x1", 1, _keys(1, [16]), np.zeros(1, np.int64),
                    _icbs_nonce_counter0(1, 1), np.array([64 * KIB], np.int64), 1)


def config2(n: int = 1000, size: int = MIB, in_flight: int = 64) -> Workload:
    """AES-128-CTR, 1 MiB payloads, 64 in flight, one key, 1,000 requests (configs[1])."""
    return Workload("c2_aes128_1MiB_x%d_w%d" % (n, in_flight), 2, _keys(2, [16]),
                    np.zeros(n, np.int64), _icbs_nonce_counter0(2, n),
                    np.full(n, size, np.int64), in_flight)


def config3(n: int = 200, size: int = 8 * MIB, in_flight: int = 16) -> Workload:
    """AES-256-CTR, 8 MiB payloads, 16 in flight, one key, 200 requests (configs[2])."""
    return Workload("c3_aes256_8MiB_x%d_w%d" % (n, in_flight), 3, _keys(3, [32]),
                    np.zeros(n, np.int64), _icbs_nonce_counter0(3, n),
                    np.full(n, size, np.int64), in_flight)


def config4(n: int = 10000, in_flight: int = 256) -> Workload:
    """Fine-grained mix (configs[3]): sizes log-uniform on 1 KiB-64 KiB, a multiple
    of 16 plus a 0-15 byte tail, per-request AES-128 or AES-256 key, fully random
    16-byte ICBs (exercises counter carries), 256 in flight."""
    rng = _rng(4, _STREAM_LENS)
    u = rng.uniform(10.0, 16.0, size=n)
    base = (np.floor(np.exp2(u) / 16.0) * 16).astype(np.int64)
    tail = rng.integers(0, 16, size=n, dtype=np.int64)
    length = np.minimum(base + tail, 64 * KIB)
    is256 = rng.integers(0, 2, size=n, dtype=np.int64)
    keys = _keys(4, [32 if b else 16 for b in is256])
    icb = _rng(4, _STREAM_ICBS).integers(0, 256, size=(n, 16), dtype=np.uint8)
    return Workload("c4_mix_1KiB-64KiB_x%d_w%d" % (n, in_flight), 4, keys,
                    np.arange(n, dtype=np.int64), icb, length, in_flight)


def fixed_size(size: int, n: int, in_flight: int, keybits: int = 128, config_index: int = 5) -> Workload:
    """One cell of the sweep (configs[4]) / the 4 KiB latency case: n requests of
    ``size`` bytes, one shared key, distinct ICBs (nonce || counter 0)."""
    return Workload("aes%d_%dB_x%d_w%d" % (keybits, size, n, in_flight), config_index,
                    _keys(config_index, [keybits // 8]), np.zeros(n, np.int64),
                    _icbs_nonce_counter0(config_index, n), np.full(n, size, np.int64), in_flight)


def edge_icbs() -> list:
    """ICBs whose low 8/32/64/128 bits are about to carry (reading R4)."""
    out = []
    for low_ones in (1, 4, 8, 12, 16):
        b = bytearray(range(0x10, 0x20))
        for k in range(low_ones):
            b[15 - k] = 0xFF
        out.append(bytes(b))
    # carries that land a few blocks into the stream rather than on the first increment
    b = bytearray(b"\xa5" * 16)
    b[12:16] = (0xFFFFFFFF - 5).to_bytes(4, "big")
    out.append(bytes(b))
    b = bytearray(b"\x5a" * 16)
    b[8:16] = (0xFFFFFFFFFFFFFFFF - 300).to_bytes(8, "big")
    out.append(bytes(b))
    out.append(((1 << 128) - 3).to_bytes(16, "big"))
    return out
