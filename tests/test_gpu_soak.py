"""-m gpu: a short randomised soak of the persistent engine -- four submitter threads, sizes 0 B .. 2 MiB with
ragged tails, AES-128/192/256, shared contexts (key-table path) and one-shot contexts (raw-key path), ICBs about to
carry, in place and out of place, a quarter of the requests in ECB-encrypt / ECB-decrypt / CBC-decrypt, a small ring
that fills up, three engine cycles with 2, 1 and 5 dispatcher warps -- every byte against the oracle."""
import threading
import time

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _worker(B, G, o, t, stop_at, errors, counts):
    rng = np.random.default_rng(260702630 + t)
    shared = [(k, B.aes_ctx_create(k)) for k in (rng.bytes(16), rng.bytes(24), rng.bytes(32))]
    try:
        while time.time() < stop_at and not errors:
            batch = []
            for _ in range(int(rng.integers(1, 40))):
                n = int(rng.integers(0, 64)) if rng.random() < 0.1 else int(2 ** rng.uniform(4, 21)) + int(rng.integers(0, 16))
                data = np.frombuffer(rng.bytes(n), dtype=np.uint8)
                icb = rng.bytes(16) if rng.random() < 0.7 else rng.bytes(12) + b"\xff\xff\xff" + bytes([int(rng.integers(0, 256))])
                if rng.random() < 0.5:
                    key, ctx = shared[int(rng.integers(0, 3))]
                    own = False
                else:
                    key = rng.bytes((16, 24, 32)[int(rng.integers(0, 3))])
                    ctx, own = B.aes_ctx_create(key), True
                mode = int(rng.integers(1, 4)) if rng.random() < 0.25 else 0   # 1 ECB-enc, 2 ECB-dec, 3 CBC-dec
                if mode:
                    n -= n % 16                                                # whole blocks only
                    data = data[:n]
                src = G.to_device(data) if n else G.device_empty(0)
                dst = src if (rng.random() < 0.3 and mode != 3) else G.device_empty(n)   # CBC-decrypt is out of place
                batch.append((key, icb, data, ctx, own, src, dst, mode))
            G.stream_sync()
            hs = []
            for key, icb, data, ctx, own, src, dst, mode in batch:
                while True:
                    try:
                        if mode == 0:
                            hs.append(B.aes_ctr_submit(ctx, icb, src.data_ptr(), dst.data_ptr(), len(data)))
                        elif mode == 3:
                            hs.append(B.aes_cbc_decrypt_submit(ctx, icb, src.data_ptr(), dst.data_ptr(), len(data)))
                        else:
                            hs.append(B.aes_ecb_submit(ctx, mode == 2, src.data_ptr(), dst.data_ptr(), len(data)))
                        break
                    except B.AesOffError as e:
                        if e.code != B.AES_E_AGAIN:
                            raise
                if own:
                    B.aes_ctx_destroy(ctx)  # allowed as soon as the submit has returned
            for h in hs:
                B.aes_wait(h, 30_000_000_000)
            for key, icb, data, ctx, own, src, dst, mode in batch:
                want = (o.ctr(key, icb, data) if mode == 0 else o.ecb_encrypt(key, data) if mode == 1 else
                        o.ecb_decrypt(key, data) if mode == 2 else o.cbc_decrypt(key, icb, data))
                if dst.cpu().numpy()[: len(data)].tobytes() != want:
                    errors.append("thread %d: mode %d, %d bytes, %d-bit key, icb %s" % (t, mode, len(data), 8 * len(key), icb.hex()))
                    return
                counts[t] += 1
    except Exception as e:  # noqa: BLE001
        errors.append("thread %d: %r" % (t, e))
    finally:
        for _, c in shared:
            B.aes_ctx_destroy(c)


def test_randomised_soak():
    import gpu_util as G
    import paper_2607_02630_b200.binding as B
    from oracle import oracle as o

    torch = G.torch_cuda()
    torch.zeros(1, device="cuda:0")
    torch.cuda.synchronize()
    errors, counts = [], [0] * 4
    for ring_slots, n_disp in ((64, 2), (0, 1), (128, 5)):
        B.aes_engine_start(0, ring_slots=ring_slots, idle_exit_ms=60000, n_dispatchers=n_disp)
        try:
            stop_at = time.time() + 3.0
            ths = [threading.Thread(target=_worker, args=(B, G, o, t, stop_at, errors, counts)) for t in range(4)]
            [x.start() for x in ths]
            [x.join() for x in ths]
        finally:
            B.aes_engine_stop()
    assert not errors, errors[:3]
    assert sum(counts) > 200
