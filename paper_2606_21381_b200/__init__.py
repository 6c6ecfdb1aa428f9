"""B200-native OSOG forward-render hot path (arxiv/paper_2606_21381): C-ABI library libosog.so + thin binding.

The names mirror include/osog.h.  Nothing here imports oracle/ (test infrastructure).
"""
from .binding import (Context, Particles, OsogError, make_optics, make_dic, make_brightfield, optics_from_scene, lib, lib_path, osog_tile_size, render_opd_static, lib_limits,
                      osog_config, osog_particles, osog_optics, osog_dic, osog_brightfield, EXPORTS,
                      OSOG_OK, OSOG_EINVAL, OSOG_ECUDA, OSOG_ECAPACITY, OSOG_ENOMEM, OSOG_ELIMIT, OSOG_WBADPARTICLE, OSOG_WOVERFLOW)

__all__ = ["Context", "Particles", "OsogError", "make_optics", "make_dic", "make_brightfield", "optics_from_scene", "lib", "lib_path", "osog_tile_size", "render_opd_static", "lib_limits",
           "osog_config", "osog_particles", "osog_optics", "osog_dic", "osog_brightfield", "EXPORTS"]
