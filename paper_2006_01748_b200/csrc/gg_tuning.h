/* gg_tuning.h -- tuning knobs of libgg.so.  NOT part of the installed interface (include/gg.h):
 * these select among compiled builds and launch shapes for re-tuning on other boxes and let the
 * tests force every build through the parity checks.  Values are passed to gg_set_option. */
#ifndef GG_TUNING_H_
#define GG_TUNING_H_

#ifdef __cplusplus
extern "C" {
#endif

enum {
    GG_OPT_STREAM_VARIANT = 3,  /* build (rows per TMA box, ring stages) of the STREAM kernel:
                                   0 .. gg_num_stream_variants()-1                                 */
    GG_OPT_ITEMS_PER_WARP = 4,  /* target work items (row chunk x tile column) per resident CTA    */
    GG_OPT_STREAM_WARPS = 5,    /* warps (= strips) per CTA: STREAM 1, 2, 4, 8; STREAM2 1, 2, 4;
                                   PAIR 1..8; 0 = from nx                                          */
    GG_OPT_STREAM2_VARIANT = 6, /* build of the STREAM2 kernel; -1 = tuned default for the dtype   */
    GG_OPT_PAIR_VARIANT = 7,    /* build of the PAIR kernel; -1 = tuned default                    */
    GG_OPT_QUAD_VARIANT = 8,    /* build of the QUAD kernel; -1 = tuned default for the dtype      */
    GG_OPT_RESIDENT_IMPL = 9,   /* GG_KERNEL_RESIDENT: 0 = one cluster per simulation where it fits
                                   (gg_cluster.cuh), 1 = always the slab kernel (gg_resident.cuh)  */
    GG_OPT_CLUSTER_CTAS = 10    /* CTAs per cluster of gg_cluster.cuh: 2, 4, 8, 16; 0 = from the batch */
};

/* number of builds selectable with the corresponding GG_OPT_*_VARIANT */
int gg_num_stream_variants(void);
int gg_num_stream2_variants(void);
int gg_num_pair_variants(void);
int gg_num_quad_variants(void);

#ifdef __cplusplus
}
#endif
#endif /* GG_TUNING_H_ */
