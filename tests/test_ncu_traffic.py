"""The helper that records roofline.traffic (paper_2509_06525_b200/ncu_traffic.py) parses ncu's raw CSV page:
matching launches are averaged, launches a capture cut short (nan) are skipped, other units are refused."""
import pytest

from paper_2509_06525_b200 import ncu_traffic


def _rows(unit="byte"):
    return [["ID", "Kernel Name", "dram__bytes_read.sum", "dram__bytes_write.sum"],
            ["", "", unit, unit],
            ["0", "void gtb::cheb_step_x2_kernel<0, 0, 3, 0>(StepArgs)", "10,000", "3000"],
            ["1", "void gtb::reduce_partials_kernel(...)", "64", "64"],
            ["2", "void gtb::cheb_step_x2_kernel<0, 0, 3, 0>(StepArgs)", "12000", "3000"],
            ["3", "void gtb::cheb_step_x2_kernel<0, 0, 3, 0>(StepArgs)", "nan", "nan"]]


def test_mean_over_matching_launches_skipping_cut_short_ones():
    value, count = ncu_traffic.dram_bytes_per_launch(_rows(), "cheb_step_x2_kernel")
    assert count == 2 and value == pytest.approx(14000.0)


def test_other_units_and_missing_kernels_are_refused():
    with pytest.raises(SystemExit):
        ncu_traffic.dram_bytes_per_launch(_rows("Gbyte"), "cheb_step_x2_kernel")
    with pytest.raises(SystemExit):
        ncu_traffic.dram_bytes_per_launch(_rows(), "cheb_tile_kernel")
