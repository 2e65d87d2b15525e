"""WorkloadSpec (cfneb_workloads) -> cfneb_params.  Marshalling only."""
from .binding import CELL_B, default_params


def params_for(spec, cell_factor=1.0, cell_mode=CELL_B, max_images=None, max_neighbors=None, **overrides):
    """cfneb_params for a BASELINE.json config: potential, FIRE constants, spring, skin, capacities."""
    kw = dict(potential=int(spec.potential), pot=list(spec.pot), k_spring=float(spec.k_spring),
              climb=int(bool(spec.climb)), cell_mode=int(cell_mode), cell_factor=float(cell_factor),
              skin=float(spec.skin), max_neighbors=int(max_neighbors or spec.max_neighbors),
              max_images=int(max_images or max(spec.max_images, spec.n_images)), fire=dict(spec.fire))
    types = getattr(spec, "types", None)
    if types is not None:
        kw["types"] = types
    kw.update(overrides)
    return default_params(**kw)
