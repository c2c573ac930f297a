"""Host logic of the scan front end (paper_1802_00147_b200/scan.py): class-change matrix and dFLI histogram of two
scans of the same grid -- the deliverable of BASELINE config 3 ("compared against QM-off on identical seeds").  CPU."""
import numpy as np

from paper_1802_00147_b200 import scan


def test_class_change_matrix_and_dfli_histogram():
    fli_a = np.array([3.0, 3.1, 6.5, 7.0, 2.9, 3.3, 9.0, 3.0])
    st_a = np.array([0, 0, 0, 0, 1, 0, 0, 0])
    fli_b = np.array([3.005, 6.2, 6.4, 3.0, 2.9, 3.3, 9.5, 2.0])
    st_b = np.array([0, 0, 0, 0, 0, 1, 0, 256])            # 256 = mode-2 skip flag: not a drop
    cmp = scan.compare_runs(dict(fli=fli_a, status=st_a), dict(fli=fli_b, status=st_b))
    assert cmp["matrix"].tolist() == [[2, 1, 1], [1, 2, 0], [1, 0, 0]]
    assert cmp["matrix"].sum() == cmp["cells"] == 8 and cmp["changed"] == 4 and cmp["live_both"] == 6
    assert cmp["dfli_hist"].sum() == 6
    d = np.array([0.005, 3.1, -0.1, -4.0, 0.5, -1.0])
    want, _ = np.histogram(d, bins=scan.DFLI_EDGES)
    assert np.array_equal(cmp["dfli_hist"], want)
    assert abs(cmp["mean_abs_dfli_regular"] - np.mean([0.005, 1.0])) < 1e-12
    text = scan.report_markdown(cmp, "QM off", "QM on", "head")
    assert "| regular | 2 | 1 | 1 |" in text and "rows = QM off" in text and text.count("\n| [") == len(scan.DFLI_EDGES) - 1


def test_classes_threshold_is_the_papers():
    assert scan.FLI_THRESHOLD == 5.8
    assert scan.classes([5.79, 5.8, 100.0, 1.0], [0, 0, 2, 3]).tolist() == [0, 1, 2, 2]
