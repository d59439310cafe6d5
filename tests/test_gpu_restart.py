"""-m gpu: engine life cycle across aes_engine_stop / aes_engine_start (own module: the engine tests
keep one engine running for the whole module)."""
import numpy as np
import pytest

from paper_2607_02630_b200 import workloads

pytestmark = pytest.mark.gpu


def test_installed_context_survives_restart():
    """A context whose key sits in the key table keeps working across aes_engine_stop/start, with the
    same ring geometry (table kept) and with another one (table rebuilt, the key is installed again)."""
    import gpu_util as G
    import paper_2607_02630_b200.binding as B
    from oracle import oracle as o

    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE, 7700]))
    key = rng.bytes(32)
    data = np.frombuffer(rng.bytes(20000), dtype=np.uint8)
    src = G.to_device(data)
    dst = G.device_empty(len(data))
    G.stream_sync()
    ctx = B.aes_ctx_create(key)
    for ring_slots in (0, 0, 256, 0):
        B.aes_engine_start(0, ring_slots=ring_slots, idle_exit_ms=60000)
        try:
            for _ in range(4):
                icb = rng.bytes(16)
                B.aes_wait(B.aes_ctr_submit(ctx, icb, src.data_ptr(), dst.data_ptr(), len(data)))
                assert dst.cpu().numpy().tobytes() == o.ctr(key, icb, data)
        finally:
            B.aes_engine_stop()
    B.aes_ctx_destroy(ctx)
