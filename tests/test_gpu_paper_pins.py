"""The paper's fully analysed map (HP 3x3x3, Table 4 :405-406) on the GPU: every number the
paper prints for it, and the survey's independent whole-map integers (tests/golden/whole_maps.txt), must come out of
the CUDA path.  The oracle cannot finish 2^27 x 103 346 evaluations in a test, so the pins are the reference here; the
oracle still checks sampled ranges."""
import numpy as np
import pytest
import torch

from oracle import gp_oracle as orc
from paper_2008_05612_b200 import gpmap
from tests._golden import read_pins, read_whole_maps

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def map_3x3x3():
    S = gpmap.Structures(3, 3, 3)
    n = 1 << S.N
    ph = torch.empty(n, dtype=torch.uint16, device="cuda")
    S.enumerate_map(ph)                                   # reversal identity, 51 704 representatives
    hist = gpmap.designability(ph, S.C).cpu().numpy().astype(np.int64)
    R, Dl, Oc, pairs = gpmap.robustness(ph, S.N, S.C)
    torch.cuda.synchronize()
    return S, ph, hist, R.cpu().numpy(), Dl.cpu().numpy(), Oc.cpu().numpy(), int(pairs)


def test_paper_printed_values(map_3x3x3):
    S, ph, hist, R, Dl, Oc, pairs = map_3x3x3
    pins = read_pins()
    n = 1 << 27
    des = hist[:S.C]
    assert S.C == pins["folds_3x3x3_classes"]
    assert int((des == 0).sum()) == pins["zero_designability_3x3x3"]
    assert int((des > 0).sum()) == pins["phenotypes_3x3x3"]
    folding = int(des.sum())
    assert round(100.0 * folding / n, 2) == pins["fold_percentage_3x3x3"]
    assert round(100.0 * int(hist[S.C]) / n, 2) == pins["deleterious_percentage_3x3x3"]
    assert int(des.max()) == 2 * pins["ns_top_fold_3x3x3"]          # N_s is printed per directed fold (R1)
    live = des > 0
    assert int((Oc[live] == 0).sum()) == pins["isolated_phenotypes_3x3x3"]
    denom = 27.0 * des[live]
    # "on average 4.0 %" (:244-248); the exact mean is 0.0407, i.e. the paper truncated
    assert abs(float((Oc[live] / denom).mean()) - pins["mean_other_fraction_3x3x3"]) < 0.001
    assert round(float((Dl[live] / denom).mean()), 4) == pins["mean_phi_del_3x3x3"]
    assert round(100.0 * (1.0 - pins["isolated_phenotypes_3x3x3"] / live.sum()), 1) == pins["connected_percent_3x3x3"]


def test_survey_whole_map_integers(map_3x3x3):
    S, ph, hist, R, Dl, Oc, pairs = map_3x3x3
    gold = read_whole_maps()["3x3x3"]
    des = hist[:S.C]
    assert int(des.sum()) == gold["folding"] and int(hist[S.C]) == gold["null"]
    assert sorted(des.tolist(), reverse=True)[:5] == gold["top5"]
    assert (int(R.sum()), int(Dl.sum()), int(Oc.sum()), pairs) == (gold["sumR"], gold["sumD"], gold["sumO"], gold["pairs"])


def test_map_path_equals_prefix_path_and_oracle_on_ranges(map_3x3x3, oracle_structures):
    S, ph, *_ = map_3x3x3
    O = oracle_structures(3, 3, 3)
    buf = torch.empty(1 << 16, dtype=torch.uint16, device="cuda")
    for begin in (0, (1 << 27) - (1 << 16), 0x2B5 << 16, 0x555 << 16):
        S.enumerate(begin, 1 << 16, buf)                  # prefix path: all 103 346 directed structures
        assert torch.equal(buf.view(torch.int16), ph[begin:begin + (1 << 16)].view(torch.int16)), begin
        want = O.enumerate(begin + 1024, 512, want_gap=False)
        assert np.array_equal(ph[begin + 1024:begin + 1536].cpu().numpy(), want), begin


def test_classes_connected_to_the_top_fold(map_3x3x3):
    """'0.86 % of phenotypes are connected to the most designable fold': 406 of 47 449."""
    S, ph, hist, R, Dl, Oc, pairs = map_3x3x3
    pins = read_pins()
    des = hist[:S.C]
    top = int(np.argmax(des))
    row = gpmap.phi_row(ph, S.N, S.C, top).cpu().numpy()
    assert int(row[top]) == int(R[top])                       # the diagonal entry is the neutral count
    connected = int(((row[:S.C] > 0) & (np.arange(S.C) != top)).sum())
    assert connected == 406
    assert round(100.0 * connected / int((des > 0).sum()), 2) == pins["connected_to_top_percent"]
