"""Mutation check of the oracle's pins.  CPU only.

Every entry of MUTATIONS is a one-line change of oracle/sf_oracle.c of the kind a plausible slip would produce
(a dropped term, a wrong sign, a wrong height or half-sample convention).  The test copies the source to a
temporary directory, applies the change (the original text must occur exactly as often as stated, so an edit of
the oracle that invalidates a mutation fails loudly here), builds it, makes the pin modules use that build, and
asserts that AT LEAST ONE of the named pins fails.  A mutation that survives means the oracle is unpinned there.

The pins named per mutation are the fast ones among those that notice it; they are called in-process as plain
functions (their parametrisation is given explicitly).
"""
import os
import subprocess

import pytest

import oracle.sf_oracle as SO

import test_oracle_dd as TD
import test_oracle_pins as T1
import test_oracle_pins2 as T2
import test_oracle_pins3 as T3
import test_oracle_recon as TR

SRC = os.path.join(os.path.dirname(os.path.abspath(SO.__file__)), "sf_oracle.c")

C4 = dict(index=4, shrink=dict(nx=12, ny=12, nz=12, nu=24, nv=24, n_views=6))

# name -> (old text, occurrences expected, which occurrence to replace, new text, [(pin, kwargs), ...])
MUTATIONS = {
    # ---- the VERDICT's table ------------------------------------------------------------------------------
    "amplitude_2d_norm_in_3d": (
        "double norm = sqrt(e[0]*e[0] + e[1]*e[1] + e[2]*e[2]);", 1, 0,
        "double norm = sqrt(e[0]*e[0] + e[1]*e[1]);",
        [(T3.test_tilted_frame_config4_shape, {})]),
    "axial_ends_at_0p45_dz": (
        "double Pm[3] = { Pc[0], Pc[1], Pc[2] - 0.5*g->dz }, Pp[3] = { Pc[0], Pc[1], Pc[2] + 0.5*g->dz };", 1, 0,
        "double Pm[3] = { Pc[0], Pc[1], Pc[2] - 0.45*g->dz }, Pp[3] = { Pc[0], Pc[1], Pc[2] + 0.45*g->dz };",
        [(T1.test_p4_golden_3d, {})]),
    "arc_row_coordinate_over_a": (
        "*t = f->R * c / sqrt(a*a + b*b) - f->Dv;", 1, 0,
        "*t = f->R * c / a - f->Dv;",
        [(T3.test_tilted_frame_footprint_from_ray_detector_intersection, dict(det="arc"))]),
    "amplitude_dy_only": (
        "*amp = norm * (rx < ry ? rx : ry);", 1, 0,
        "*amp = norm * ry;",
        [(T1.test_p2_hand_worked_2d, {}), (T3.test_tilted_frame_config4_shape, {})]),
    "dd_face_inverted": (
        "int along_y = g->dy * ex <= g->dx * ey;", 1, 0,
        "int along_y = g->dy * ex > g->dx * ey;",
        [(TD.test_dd_hand_worked_2d, {})]),
    "corners_at_lower_face_instead_of_mid_plane": (
        "double P[3] = { Pc[0] + sx*0.5*g->dx, Pc[1] + sy*0.5*g->dy, Pc[2] };", 1, 0,
        "double P[3] = { Pc[0] + sx*0.5*g->dx, Pc[1] + sy*0.5*g->dy, Pc[2] - 0.5*g->dz };",
        [(T3.test_tilted_frame_footprint_from_ray_detector_intersection, dict(det="flat"))]),
    "frame_normal_never_flipped": (
        "if (dot3(DS, n) < 0.0) { n[0] = -n[0]; n[1] = -n[1]; n[2] = -n[2]; }", 1, 0,
        "",
        [(T3.test_reversed_channel_axis_mirrors_the_projections, C4)]),
    "recon_arc_taps_use_the_flat_formula": (
        "else { double sn = PI * f.R * sin(n*g->du / f.R); h = -1.0 / (sn*sn); }", 1, 0,
        "else { double sn = PI * n*g->du; h = -1.0 / (sn*sn); }",
        [(TR.test_fan_beam_fbp_of_a_wide_disk_on_the_arc_detector, {})]),
    "recon_arc_depth_weight_over_a2": (
        "sqrt(Sn*Sn + Su*Su) * f->R / (a*a + b*b);", 1, 0,
        "sqrt(Sn*Sn + Su*Su) * f->R / (a*a);",
        [(TR.test_fan_beam_fbp_of_a_far_off_axis_disk, dict(det="arc"))]),
    "recon_arc_preweight_without_cos_gamma": (
        "pw[k] = p[k] * cos(uk / f.R) * f.R / sqrt(f.R*f.R + t*t);", 1, 0,
        "pw[k] = p[k] * f.R / sqrt(f.R*f.R + t*t);",
        [(TR.test_fan_beam_fbp_of_a_far_off_axis_disk, dict(det="arc"))]),
    "recon_flat_preweight_without_t2": (
        "pw[k] = p[k] * f.R / sqrt(f.R*f.R + s*s + t*t);", 1, 0,
        "pw[k] = p[k] * f.R / sqrt(f.R*f.R + s*s);",
        [(TR.test_fdk_of_a_z_invariant_cylinder_off_the_mid_plane, dict(det="flat"))]),
    # ---- further slips of the same kind ------------------------------------------------------------------
    "recon_flat_preweight_without_s2": (
        "pw[k] = p[k] * f.R / sqrt(f.R*f.R + s*s + t*t);", 1, 0,
        "pw[k] = p[k] * f.R / sqrt(f.R*f.R + t*t);",
        [(TR.test_fan_beam_fbp_of_a_far_off_axis_disk, dict(det="flat"))]),
    "recon_arc_preweight_without_row_cosine": (
        "pw[k] = p[k] * cos(uk / f.R) * f.R / sqrt(f.R*f.R + t*t);", 1, 0,
        "pw[k] = p[k] * cos(uk / f.R);",
        [(TR.test_fdk_of_a_z_invariant_cylinder_off_the_mid_plane, dict(det="arc"))]),
    "recon_flat_depth_weight_uses_R_for_d": (
        "(-Sn) * f->R / (a*a)", 1, 0,
        "f->R * f->R / (a*a)",
        [(TR.test_recon_backprojection_weights_are_normalised, dict(algo="SF"))]),
    "recon_sumF1_is_the_full_base": (
        "double sumF1 = 0.5*(tau[3] + tau[2] - tau[1] - tau[0]) / g->du", 1, 0,
        "double sumF1 = (tau[3] - tau[0]) / g->du",
        [(TR.test_recon_backprojection_weights_are_normalised, dict(algo="SF"))]),
    "recon_filter_not_scaled_by_du": (
        "q[k] = g->du * acc;", 1, 0,
        "q[k] = acc;",
        [(TR.test_fan_beam_fbp_of_a_wide_disk_on_the_arc_detector, {})]),
    "trapezoid_cdf_falling_ramp_sign": (
        "+ (s - t2) - (s - t2)*(s - t2) / (2.0*(t3 - t2));", 1, 0,
        "+ (s - t2) + (s - t2)*(s - t2) / (2.0*(t3 - t2));",
        [(T1.test_p1_trap_cdf_vs_quadrature, {})]),
    "cell_centre_half_sample": (
        "double uk = (k - 0.5*(g->nu - 1))*g->du;\n        F1", 1, 0,
        "double uk = (k - 0.5*g->nu)*g->du;\n        F1",
        [(T1.test_p2_hand_worked_2d, {})]),
    "voxel_centre_half_sample": (
        "double Pc[3] = { g->ox + (ix - 0.5*(g->nx - 1))*g->dx,\n", 1, 0,
        "double Pc[3] = { g->ox + (ix - 0.5*g->nx)*g->dx,\n",
        [(T1.test_p2_hand_worked_2d, {})]),
    "flat_detector_offset_sign": (
        "*s = f->R * b / a - f->Du;", 1, 0,
        "*s = f->R * b / a + f->Du;",
        [(T3.test_tilted_frame_config4_shape, {})]),
    "row_offset_sign": (
        "*t = f->R * c / a - f->Dv;", 1, 0,
        "*t = f->R * c / a + f->Dv;",
        [(T3.test_tilted_frame_config4_shape, {})]),
    "arc_angle_arguments_swapped": (
        "*s = f->R * atan2(b, a);", 1, 0,
        "*s = f->R * atan2(a, b);",
        [(T1.test_p3_golden_2d, {})]),
    "F2_not_divided_by_dv": (
        "F2[l - llo] = (hi - lo > 0.0 ? hi - lo : 0.0) / g->dv;", 1, 0,
        "F2[l - llo] = (hi - lo > 0.0 ? hi - lo : 0.0);",
        [(T1.test_p4_golden_3d, {})]),
    # ---- the three that survived ---------------------------------------------------------
    "sftt_half_chord_0p4": (
        "double P[3] = { Pc[0] + sn*0.5*lth*ux, Pc[1] + sn*0.5*lth*uy, Pc[2] + sz*0.5*g->dz };", 1, 0,
        "double P[3] = { Pc[0] + sn*0.4*lth*ux, Pc[1] + sn*0.4*lth*uy, Pc[2] + sz*0.5*g->dz };",
        [(T3.test_sftt_axial_profile_is_the_chord_fraction_between_the_voxel_faces, {}),
         (T3.test_sftt_footprint_from_ray_detector_intersection, dict(det="flat"))]),
    "sftt_recon_normalised_by_the_base": (
        "if (sumF2_out) *sumF2_out = 0.5*(xi[3] + xi[2] - xi[1] - xi[0]) / g->dv;", 1, 0,
        "if (sumF2_out) *sumF2_out = (xi[3] - xi[0]) / g->dv;",
        [(TR.test_recon_backprojection_weights_are_normalised, dict(algo="SF-TT"))]),
    "dd_tie_goes_the_other_way": (
        "int along_y = g->dy * ex <= g->dx * ey;", 1, 0,
        "int along_y = g->dy * ex < g->dx * ey;",
        [(TD.test_dd_exact_tie_takes_the_face_across_y, {})]),
    "sftt_chord_of_the_longer_axis": (
        "double lth = rx_ < ry_ ? rx_ : ry_;", 1, 0,
        "double lth = rx_ < ry_ ? ry_ : rx_;",
        [(T3.test_sftt_footprint_from_ray_detector_intersection, dict(det="arc"))]),
    "backprojection_drops_the_amplitude": (
        "acc += amp * F1[k - klo] * F2[l - llo] * y[(size_t)l*g->nu + k];", 1, 0,
        "acc += F1[k - klo] * F2[l - llo] * y[(size_t)l*g->nu + k];",
        [(T2.test_p13_dense_matrix, dict(det="flat"))]),
}


def _build_mutant(tmp_path, name):
    old, count, which, new, _ = MUTATIONS[name]
    text = open(SRC).read()
    assert text.count(old) == count, "mutation %r no longer matches oracle/sf_oracle.c (%d occurrences)" % (
        name, text.count(old))
    pos = -1
    for _ in range(which + 1):
        pos = text.index(old, pos + 1)
    text = text[:pos] + new + text[pos + len(old):]
    c = tmp_path / (name + ".c")
    so = tmp_path / (name + ".so")
    c.write_text(text)
    subprocess.check_call(["gcc", "-O1", "-fopenmp", "-shared", "-fPIC", "-o", str(so), str(c), "-lm"])
    return SO.load_library(str(so))


@pytest.mark.parametrize("name", sorted(MUTATIONS))
def test_mutation_is_caught(name, tmp_path, monkeypatch):
    SO._load()                                   # the true build, loaded before it is shadowed
    mutant = _build_mutant(tmp_path, name)
    monkeypatch.setattr(SO, "_lib", mutant)
    killed = []
    for pin, kwargs in MUTATIONS[name][4]:
        try:
            pin(**kwargs)
        except Exception:                        # an assertion, or the pin tripping over a missing footprint
            killed.append(pin.__name__)
            break
    assert killed, "mutation %r survives its pins: the oracle is unpinned there" % name


def test_the_unmutated_oracle_passes_the_named_pins():
    """Guards the guard: every pin used above is green on the real oracle (so a failure above is the mutation's)."""
    SO._load()
    seen = set()
    for _, _, _, _, pins in MUTATIONS.values():
        for pin, kwargs in pins:
            key = (pin.__name__, tuple(sorted((k, str(v)) for k, v in kwargs.items())))
            if key not in seen:
                seen.add(key)
                pin(**kwargs)
