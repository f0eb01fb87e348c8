"""qld_probe_read (the read-only ceiling bench.py quotes): the probe must really load every word it is charged
with -- its per-CTA checksums add up to the checksum of the whole buffer, computed here with numpy -- or the bandwidth derived
from its run time would mean nothing.  (A measuring stick, not a step of the method: there is no oracle function for it.)"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n_bytes", [16, 16 * 1000 + 7, (1 << 24) + 48, 3 * (1 << 24) + 16 * 12345])
def test_probe_reads_every_word(n_bytes):
    import torch
    from paper_1511_03390_b200 import qld
    rng = np.random.default_rng(n_bytes)
    host = rng.integers(0, 256, size=n_bytes, dtype=np.uint8)
    out = qld.probe_read(torch.from_numpy(host).cuda())
    torch.cuda.synchronize()
    w = host[: n_bytes // 16 * 16].view(np.uint32).reshape(-1, 4)
    want = int((w[:, 0] ^ w[:, 1] ^ w[:, 2] ^ w[:, 3]).astype(np.uint64).sum() % (1 << 32))
    got = int(out.cpu().numpy().view(np.uint32).astype(np.uint64).sum() % (1 << 32))
    assert got == want


def test_probe_rejects_bad_arguments():
    import torch
    from paper_1511_03390_b200 import qld
    buf = torch.zeros(64, dtype=torch.uint8, device="cuda")
    with pytest.raises(qld.QLDError):
        qld.probe_read(buf[1:33])                              # not 16-byte aligned
    with pytest.raises(qld.QLDError):
        qld.probe_read(buf[:8])                                # less than one word
