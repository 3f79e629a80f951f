"""paper_2606_00817_b200 - B200-native batched Directed Distance Field queries.

Thin Python binding (argument marshalling only) over the C ABI in include/ddf.h; every step of
the path runs in the CUDA kernels of csrc/.  torch is used for device memory and streams only.
There is no CPU fallback: importing works anywhere, calling needs libddf.so and a B200.
"""
from .binding import (  # noqa: F401
    DdfError, DdfLayout, DdfCamera, DdfScene, SdfTraceParams, Model, lib, lib_path,
    ddf_create, ddf_destroy, ddf_query, ddf_query_host, ddf_query_logits, ddf_query_ao, ddf_set_path,
    ddf_get_info, ddf_camera_from_seed, ddf_gen_camera, ddf_gen_sphere_points, ddf_gen_shadow,
    ddf_gen_gbuffer, ddf_gen_ao, ddf_ao_reduce, ddf_shadow_test, sdf_sphere_trace, ddf_status_string,
    DdfHashgridLayout, make_hashgrid_layout, ddf_hashgrid_table_entries, ddf_create_hashgrid,
    ddf_gen_shadow_from_hits, ddf_gen_shadow_from_hits_static, STATIC_MAX_RAYS, ddf_query_shadowed, ddf_query_shadowed_lights, ddf_gen_ao_from_hits, ddf_query_ao_wavefront, ddf_query_shaded, ddf_query_ao_points,
    DdfTrainParams, make_train_params, Trainer, ddf_trainer_create, ddf_trainer_destroy, ddf_trainer_step,
    ddf_trainer_loss_grads, ddf_trainer_export, ddf_trainer_steps, ddf_scene_raycast, ddf_gen_train_batch,
    ddf_query_camera, ddf_reserve, RESERVE_HOST, RESERVE_RAYS, RESERVE_TRACE, RESERVE_WAVE, RESERVE_ALL,
    EXPORTED_SYMBOLS,
)
from .build import build  # noqa: F401
