"""Host logic of the product: every hand-written per-element adjoint (paper_2606_04206_b200/csrc/rod_adj.cuh) against
central finite differences of its forward operator (rod_ops.cuh), compiled for the CPU in double.  This exercises the
product's own operator code (not the oracle); the warp-level data movement around it is covered by the -m gpu tests."""
import os
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_every_operator_adjoint_matches_finite_differences(tmp_path):
    exe = str(tmp_path / "adj_check")
    subprocess.run(["g++", "-std=c++17", "-O1", "-I", os.path.join(ROOT, "paper_2606_04206_b200", "csrc"), "-o", exe,
                    os.path.join(ROOT, "tests", "host", "adj_check.cpp")], check=True)
    out = subprocess.run([exe], check=True, capture_output=True, text=True).stdout
    assert "not penetrating" not in out and "inactive!" not in out, out
    rows = [l.split() for l in out.strip().splitlines()]
    assert len(rows) >= 40
    names = {r[0].rstrip("_0123456789") for r in rows}
    for need in ("bend_element", "material_curvature", "frame_update", "plasticity_active", "project_edge", "closest_points",
                 "contact", "friction_capped", "friction_stick", "rigid_response", "sdf_type", "sdf_capsule_endpoints",
                 "rodrigues", "body_point_velocity+make_pose"):
        assert need in names, need
    for name, err in rows:
        assert float(err) < 1e-6, (name, err)
