"""-m gpu: the instruction-rate microbenchmarks quoted in DESIGN.md section 7 / profiles/ run from tracked code and land
where the notes say (loose brackets: they are measurements of this GPU, not contracts)."""
import pytest

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def test_microbench_brackets():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2606_24033_b200 as P
    vals = {}
    for i in range(P.MICROBENCH_COUNT):
        name, v = P.microbench(i, 12)
        assert v > 0, name
        vals[i] = v
    assert 0.4 < vals[0] < 0.55                    # PRMT: half rate
    assert 0.4 < vals[1] < 0.55 and 0.4 < vals[2] < 0.55   # LOP3, SHF: the same pipe ...
    assert vals[8] < 0.6 and vals[9] < 0.6         # ... and they do not overlap with PRMT
    assert vals[10] > 0.75 and vals[11] > 0.7      # IMAD and HFMA2 issue beside PRMT
    assert vals[6] > 0.8                           # IADD at full rate
    assert vals[17] < vals[16]                     # byte planes are cheaper to unpack than fp16 fragments
    assert vals[18] > 30 and vals[20] < vals[18] / 2.5     # one thread issues a tcgen05.mma every ~60 clocks; issuers scale
