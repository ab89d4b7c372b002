"""Host-only front-end for the LHAPDF6 text layout: files written
by workloads.write_* are read back bit for bit through the C-ABI parser; malformed files are
refused with the documented codes.  No device is touched."""
import os

import numpy as np
import pytest

from paper_2009_06635_b200 import binding as B, build, workloads as W


@pytest.fixture(scope="module", autouse=True)
def _lib():
    build.build()
    B.lib()


def test_member_file_round_trip(tmp_path):
    spec = W.grid_nnpdf_shaped()
    p = tmp_path / "synth_0000.dat"
    W.write_lhagrid(spec, str(p))
    x, off, q, pids, vals = B.lhagrid_read(str(p))
    assert np.array_equal(x, spec.x_knots) and np.array_equal(q, spec.q_knots)
    assert np.array_equal(off, spec.q_offsets) and np.array_equal(pids, spec.pids)
    assert np.array_equal(vals, spec.values)        # repr() round-trips doubles exactly


def test_metadata_alphas_and_members(tmp_path):
    a = W.make_alphas_grid()
    p = tmp_path / "synth.info"
    W.write_lhapdf_info(str(p), 7, W.PIDS_11, a)
    q, v = B.lhapdf_info_alphas(str(p))
    assert np.array_equal(q, a.q_knots) and np.array_equal(v, a.alphas)   # incl. the list split over two lines
    assert B.lhapdf_info_members(str(p)) == 7
    (tmp_path / "nomembers.info").write_text("AlphaS_Qs: [1.0, 2.0]\nAlphaS_Vals: [0.3, 0.2]\n")
    assert B.lhapdf_info_members(str(tmp_path / "nomembers.info")) == 1


def test_tolerates_crlf_blank_lines_and_missing_trailing_separator(tmp_path):
    spec = W.grid_config1()
    p = tmp_path / "a.dat"
    W.write_lhagrid(spec, str(p))
    txt = p.read_text()
    assert txt.endswith("---\n")
    (tmp_path / "b.dat").write_text(txt[:-4].replace("\n", "\r\n") + "\r\n\r\n")
    got = B.lhagrid_read(str(tmp_path / "b.dat"))
    assert np.array_equal(got[4], spec.values) and np.array_equal(got[0], spec.x_knots)


@pytest.mark.parametrize("mutate, code", [
    (lambda t: t.replace("---\n", "", 1).replace("---\n", ""), B.PDFB_EFORMAT),         # no separator at all
    (lambda t: "\n".join(t.split("\n")[:-5]) + "\n---\n", B.PDFB_EFORMAT),              # value rows missing
    (lambda t: t.replace(t.split("\n")[6], t.split("\n")[6] + " 1.0", 1), B.PDFB_EFORMAT),  # a row with a wrong count
    (lambda t: t.replace(t.split("\n")[7], "0.1 abc 0.3", 1), B.PDFB_EFORMAT),           # not a number
])
def test_malformed_member_files(tmp_path, mutate, code):
    spec = W.grid_config1()
    p = tmp_path / "a.dat"
    W.write_lhagrid(spec, str(p))
    (tmp_path / "bad.dat").write_text(mutate(p.read_text()))
    with pytest.raises(B.PdfbError) as e:
        B.lhagrid_read(str(tmp_path / "bad.dat"))
    assert e.value.code == code


def test_missing_file_and_mismatched_blocks(tmp_path):
    with pytest.raises(B.PdfbError) as e:
        B.lhagrid_read(str(tmp_path / "nope.dat"))
    assert e.value.code == B.PDFB_EIO
    with pytest.raises(B.PdfbError) as e:
        B.lhapdf_info_alphas(str(tmp_path / "nope.info"))
    assert e.value.code == B.PDFB_EIO
    # second block on other x knots: refused (this library wants one x-knot array)
    spec = W.grid_nnpdf_shaped()
    p = tmp_path / "a.dat"
    W.write_lhagrid(spec, str(p))
    blocks = p.read_text().split("---\n")
    lines = blocks[2].split("\n")
    lines[0] = lines[0].replace(lines[0].split(" ")[1], repr(float(spec.x_knots[1]) * 1.0001), 1)
    blocks[2] = "\n".join(lines)
    (tmp_path / "bad.dat").write_text("---\n".join(blocks))
    with pytest.raises(B.PdfbError) as e:
        B.lhagrid_read(str(tmp_path / "bad.dat"))      # the one-x-array reader says which API takes the file
    assert e.value.code == B.PDFB_EXKNOTS
    assert not B.lhagrid_read_xs(str(tmp_path / "bad.dat"))[6]
    # a member file whose sub-grids have x-knot arrays of different LENGTHS (as LHAPDF allows) round-trips
    # through the *_xs reader into pdf_grid_load_xs's arguments
    xs = [spec.x_knots, W._geomspace(1e-9, 1.0, 80), spec.x_knots[::3].copy(), W._geomspace(1e-9, 1.0, 120)]
    sx = W.make_pdf_grid_xs(xs, (1.65, (1.65 * 4.92) ** 0.5, 4.92, 172.5, 1.0e5), (7, 14, 23, 20), W.PIDS_11)
    W.write_lhagrid(sx, str(tmp_path / "perx.dat"))
    xoff, x, qoff, q, pids, vals, shared = B.lhagrid_read_xs(str(tmp_path / "perx.dat"))
    assert not shared and np.array_equal(xoff, sx.x_offsets) and np.array_equal(x, sx.x_knots)
    assert np.array_equal(qoff, sx.q_offsets) and np.array_equal(q, sx.q_knots) and np.array_equal(vals, sx.values)
    # a shared-x file through the same reader
    W.write_lhagrid(spec, str(tmp_path / "shared.dat"))
    r = B.lhagrid_read_xs(str(tmp_path / "shared.dat"))
    assert r[6] and np.array_equal(r[1], np.tile(spec.x_knots, spec.n_sub)) and np.array_equal(r[5], spec.values)
    # sub-grids with different PID lists: well-formed, refused with the distinct code
    blocks = (tmp_path / "perx.dat").read_text().split("---\n")
    lines = blocks[2].split("\n")
    lines[2] = lines[2].replace("21", "22")
    blocks[2] = "\n".join(lines)
    (tmp_path / "pids.dat").write_text("---\n".join(blocks))
    with pytest.raises(B.PdfbError) as e:
        B.lhagrid_read_xs(str(tmp_path / "pids.dat"))
    assert e.value.code == B.PDFB_EXKNOTS
    # ... while a file cut short is a malformed file
    txt = (tmp_path / "perx.dat").read_text().split("\n")
    (tmp_path / "perx_cut.dat").write_text("\n".join(txt[: len(txt) // 2]) + "\n")
    with pytest.raises(B.PdfbError) as e:
        B.lhagrid_read_xs(str(tmp_path / "perx_cut.dat"))
    assert e.value.code == B.PDFB_EFORMAT
